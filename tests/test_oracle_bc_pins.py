"""Pins (-m "not gpu") for the oracle pieces the paper leaves to a reading (U13, U14, U16, U17): the wall
node extrapolation, the side selection of the subsonic far field, the CFL time step and the residual sum.  Each is
checked against what the mathematics fixes (polynomial exactness of the one-sided closure, the Riemann invariants
and the upwind side's entropy / tangential velocity, a hand formula on a Cartesian grid, the plain sum of squares),
never against the oracle's own formula or the CUDA path."""
import numpy as np
import pytest

NG = 6
GAMMA = 1.4


def _bc_box(W, n, L, q0, qinf, lo_type, hi_type, warp=0.0, viscous=0, mach=0.3):
    """Box, periodic in xi and zeta, physical faces on -eta (face 2) and +eta (face 3)."""
    X, Y, Z = W._uniform_nodes(n, L)
    xyz = np.stack([X + warp * np.sin(np.pi * Y / L[1]), Y, Z + 0.5 * warp * np.sin(2 * np.pi * X / L[0])])
    faces = [f for f in W.periodic_faces(0, L) if f["face"] not in (2, 3)]
    for s, t in ((2, lo_type), (3, hi_type)):
        faces.append(dict(block=0, face=s, type=t, nbr_block=-1, nbr_face=-1, perm=[0, 1, 2], sign=[1, 1, 1], shift=[0.0] * 3))
    prm = W.default_params(viscous=viscous, mach=mach, q_inf=qinf)
    return W.Case("bcbox", [n], [xyz], [q0], faces, prm, dt=0.0, steps=0), xyz


def _prims(q):
    rho = q[0]
    vel = q[1:4] / rho
    p = (GAMMA - 1) * (q[4] - 0.5 * rho * (vel ** 2).sum(0))
    return rho, vel, p


# ------------------------------------------------------------------------------------------------
# U13: wall node values p0, T0 = (48 a1 - 36 a2 + 16 a3 - 3 a4)/25, the 4th-order one-sided da/dn = 0
# ------------------------------------------------------------------------------------------------
def test_wall_node_extrapolation_is_exact_for_quartics_without_linear_term(po, W):
    """The 5-point one-sided first derivative (-25, 48, -36, 16, -3)/12 is exact for polynomials of degree <= 4, so
    with a(j) = c0 + c2 j^2 + c3 j^3 + c4 j^4 (zero slope at the wall) normal to the wall the closure da/dn = 0 must
    return a(0) = c0 exactly -- for p and for T separately (adiabatic wall), with rho0 = gamma p0 / T0 and zero
    momentum.  Any other weights summing to one (or a3, a4 exchanged) miss c0 at O(1)."""
    n = (8, 12, 6)
    L = (1.0, 1.5, 0.75)
    X, Y, Z = W._uniform_nodes(n, L)
    jj = np.arange(n[1], dtype=float)[None, :, None] + 0 * X  # node index normal to the wall (eta)
    # tangentially varying coefficients so that a transposed tangential index would show
    cp0 = 0.7 + 0.05 * np.sin(2 * np.pi * X / L[0]) * np.cos(2 * np.pi * Z / L[2])
    cT0 = 1.1 + 0.04 * np.cos(2 * np.pi * X / L[0])
    p = cp0 + 3e-3 * jj ** 2 - 4e-4 * jj ** 3 + 2.5e-5 * jj ** 4
    T = cT0 - 2e-3 * jj ** 2 + 5e-4 * jj ** 3 - 1.5e-5 * jj ** 4
    rho = GAMMA * p / T
    rng = np.random.default_rng(7)
    u, v, w = (0.2 * rng.uniform(-1, 1, X.shape) for _ in range(3))  # velocities must not enter p0, T0
    q0 = W.prim_to_cons(rho, u, v, w, p)
    qinf = W.prim_to_cons(1.0, 0.0, 0.0, 0.0, 1 / GAMMA)
    case, _ = _bc_box(W, n, L, q0, qinf, W.WALL, W.FARFIELD)
    o = po.Oracle(case.dims, case.faces, case.params)
    o.load_case(case)  # metrics, ghost fill, apply_bc
    q = o.interior(0, "q")
    rho_w, vel_w, p_w = _prims(q[:, :, 0, :])
    T_w = GAMMA * p_w / rho_w
    assert np.abs(p_w - cp0[:, 0, :]).max() < 1e-13
    assert np.abs(T_w - cT0[:, 0, :]).max() < 1e-13
    assert np.all(q[1:4, :, 0, :] == 0.0)
    # sanity of the pin itself: the naive copy a0 = a1 and the swapped weights miss c0 by far more than the tolerance
    a = p[:, 1:5, :]
    swapped = (48 * a[:, 0] - 36 * a[:, 1] - 3 * a[:, 2] + 16 * a[:, 3]) / 25
    assert np.abs(swapped - cp0[:, 0, :]).max() > 1e-3 and np.abs(a[:, 0] - cp0[:, 0, :]).max() > 1e-3


# ------------------------------------------------------------------------------------------------
# U14: characteristic far field, subsonic branches with DISTINCT interior and far-field states
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind", ["outflow", "inflow"])
def test_farfield_subsonic_takes_each_characteristic_from_its_upwind_side(po, W, kind):
    """Along the outward normal n: the outgoing invariant R+ = u.n + 2c/(g-1) comes from the interior neighbour, the
    incoming R- = u.n - 2c/(g-1) from q_inf; entropy p/rho^g and tangential velocity come from the interior when
    the boundary normal velocity is outward (outflow) and from q_inf when it is inward (inflow)."""
    n = (10, 12, 8)
    L = (2.0, 2.4, 1.6)
    X, Y, Z = W._uniform_nodes(n, L)
    rng = np.random.default_rng(11)
    # mean flow along +y at Mach ~0.35: face 3 (+eta) is a subsonic outflow, face 2 (-eta) a subsonic inflow
    rho = 1.0 + 0.01 * rng.uniform(-1, 1, X.shape)
    u = 0.10 + 0.03 * rng.uniform(-1, 1, X.shape)
    v = 0.35 + 0.03 * rng.uniform(-1, 1, X.shape)
    w = -0.05 + 0.03 * rng.uniform(-1, 1, X.shape)
    p = (1 / GAMMA) * (1 + 0.01 * rng.uniform(-1, 1, X.shape))
    q0 = W.prim_to_cons(rho, u, v, w, p)
    qinf = W.prim_to_cons(0.8, 0.2, 0.30, 0.07, 0.8 / GAMMA)  # same c (keeps V_n's sign), entropy 0.78 vs ~0.71, other tangential / normal velocity
    case, _ = _bc_box(W, n, L, q0, qinf, W.FARFIELD, W.FARFIELD, warp=0.03)
    o = po.Oracle(case.dims, case.faces, case.params)
    o.load_case(case)
    q = o.interior(0, "q")
    kh = o.interior(0, "khat").reshape(3, 3, *q.shape[1:])
    jb, ji, sgn = (n[1] - 1, n[1] - 2, 1.0) if kind == "outflow" else (0, 1, -1.0)
    kn = kh[1][:, :, jb, :]                       # khat^eta at the boundary node
    nrm = sgn * kn / np.sqrt((kn ** 2).sum(0))    # outward unit normal
    rb, vb, pb = _prims(q[:, :, jb, :])
    ri, vi, pi = _prims(q[:, :, ji, :])
    rf, vf, pf = _prims(qinf[:, None, None] + 0 * q[:, :, jb, :])
    c = lambda r_, p_: np.sqrt(GAMMA * p_ / r_)
    un = lambda v_: (v_ * nrm).sum(0)
    g1 = GAMMA - 1
    assert np.abs(un(vb)).max() < c(rb, pb).min()             # subsonic at the boundary
    assert (sgn * vb[1] > 0).all() if kind == "outflow" else (un(vb) < 0).all()
    assert np.abs((un(vb) + 2 * c(rb, pb) / g1) - (un(vi) + 2 * c(ri, pi) / g1)).max() < 1e-13   # R+ from the interior
    assert np.abs((un(vb) - 2 * c(rb, pb) / g1) - (un(vf) - 2 * c(rf, pf) / g1)).max() < 1e-13   # R- from q_inf
    ru, vu, pu = (ri, vi, pi) if kind == "outflow" else (rf, vf, pf)   # the upwind side
    rd, vd, pd = (rf, vf, pf) if kind == "outflow" else (ri, vi, pi)   # the other side
    ent = lambda r_, p_: p_ / r_ ** GAMMA
    tang = lambda v_: v_ - un(v_) * nrm
    assert np.abs(ent(rb, pb) / ent(ru, pu) - 1).max() < 1e-13
    assert np.abs(tang(vb) - tang(vu)).max() < 1e-13
    # the pin discriminates: the other side's entropy / tangential velocity are far away
    assert np.abs(ent(rb, pb) / ent(rd, pd) - 1).min() > 1e-2
    assert np.abs(tang(vb) - tang(vd)).max() > 1e-2
    # ghosts copy the boundary node
    f = o.field(0, "q")
    for g in range(1, NG + 1):
        jg = NG + jb + (g if kind == "outflow" else -g)
        assert np.array_equal(f[:, NG:-NG, jg, NG:-NG], f[:, NG:-NG, NG + jb, NG:-NG])


# ------------------------------------------------------------------------------------------------
# U16: CFL time step on a stretched Cartesian grid, by hand
# ------------------------------------------------------------------------------------------------
def test_cfl_dt_against_hand_formula_on_a_cartesian_grid(po, W):
    """Uniform Cartesian spacings (hx, hy, hz): J khat^xi = (1/hx, 0, 0) etc., so
    dt = CFL / max_i [ |u|/hx + |v|/hy + |w|/hz + c (1/hx + 1/hy + 1/hz) ]."""
    n = (8, 10, 12)
    L = (4.0, 2.5, 24.0)
    X, Y, Z = W._uniform_nodes(n, L)
    rng = np.random.default_rng(21)
    rho = 1.0 + 0.2 * rng.uniform(-1, 1, X.shape)
    u, v, w = 0.6 * rng.uniform(-1, 1, X.shape), 0.4 * rng.uniform(-1, 1, X.shape), 1.5 * rng.uniform(-1, 1, X.shape)
    p = (1 / GAMMA) * (1 + 0.2 * rng.uniform(-1, 1, X.shape))
    q0 = W.prim_to_cons(rho, u, v, w, p)
    case = W.Case("cart", [n], [np.stack([X, Y, Z])], [q0], W.periodic_faces(0, L), W.default_params(), dt=0.0, steps=0)
    o = po.Oracle(case.dims, case.faces, case.params)
    o.load_case(case)
    hx, hy, hz = (L[a] / n[a] for a in range(3))
    c = np.sqrt(GAMMA * p / rho)
    s = np.abs(u) / hx + np.abs(v) / hy + np.abs(w) / hz + c * (1 / hx + 1 / hy + 1 / hz)
    for cfl in (0.5, 1.3):
        assert abs(o.cfl_dt(cfl) / (cfl / s.max()) - 1) < 1e-13
    # uniform state: closed form
    q1 = W.prim_to_cons(1.0 + 0 * X, 0.3 + 0 * X, -0.2 + 0 * X, 0.1 + 0 * X, 1 / GAMMA + 0 * X)
    o.interior(0, "q")[...] = q1
    want = 0.7 / (0.3 / hx + 0.2 / hy + 0.1 / hz + 1.0 * (1 / hx + 1 / hy + 1 / hz))
    assert abs(o.cfl_dt(0.7) / want - 1) < 1e-13


# ------------------------------------------------------------------------------------------------
# U17: the stage-1 residual is the plain sum of squares of the oracle's own R field
# ------------------------------------------------------------------------------------------------
def test_residual_is_the_sum_of_squares_of_r_over_all_blocks(po, W):
    case = W.c4_multiblock(nb=8, mach=0.3)
    o = po.Oracle(case.dims, case.faces, case.params)
    o.load_case(case)
    o.rhs()
    want = sum((o.interior(b, "r").astype(np.longdouble) ** 2).sum(axis=(1, 2, 3)) for b in range(len(case.dims)))
    q_before = [o.interior(b, "q").copy() for b in range(len(case.dims))]
    r_field = [o.interior(b, "r").copy() for b in range(len(case.dims))]
    dt = 1e-3
    res = o.rk_stage(1, dt, want_res=True)
    assert np.abs(res / want.astype(float) - 1).max() < 1e-14
    assert (res > 0).all()
    # and stage 1 of Eq. 20 is Q + dt R with Q^n saved
    for b in range(len(case.dims)):
        assert np.array_equal(o.interior(b, "qn"), q_before[b])
        assert np.abs(o.interior(b, "q") - (q_before[b] + dt * r_field[b])).max() < 1e-15


# ------------------------------------------------------------------------------------------------
# U17a: "summation of all inner grid points" -- the node planes a physical BC owns are not inner points
# ------------------------------------------------------------------------------------------------
def test_residual_leaves_out_the_node_planes_the_physical_bcs_own(po, W):
    """Cylinder block: WALL on the node plane j = 0, FARFIELD on j = nj-1, periodic in xi and zeta.  The stage-1 residual
    must be the sum of R_m^2 over j = 1 .. nj-2 only (computed here from the oracle's own R field in extended precision),
    and must NOT be the sum over all nodes (the two planes carry a visible share of it); Eq. 20 itself still advances every
    node (the BC overwrites the two planes afterwards)."""
    case = W.c5_cylinder(ni=32, nj=14, nk=8, ratio=1.2, r_out=8.0, noise=1e-2)
    o = po.Oracle(case.dims, case.faces, case.params)
    o.load_case(case)
    o.rhs()
    R = o.interior(0, "r").astype(np.longdouble)   # [5, k, j, i]
    inner = (R[:, :, 1:-1, :] ** 2).sum(axis=(1, 2, 3)).astype(float)
    everything = (R ** 2).sum(axis=(1, 2, 3)).astype(float)
    q0, r0 = o.interior(0, "q").copy(), o.interior(0, "r").copy()
    res = o.rk_stage(1, 1e-3, want_res=True)
    assert np.abs(res / inner - 1).max() < 1e-14
    assert np.abs(res / everything - 1).max() > 1e-3      # a dropped mask would fail here
    assert np.abs(o.interior(0, "q") - (q0 + 1e-3 * r0)).max() < 1e-15   # all nodes advanced, BC planes included

