"""Block-level pins for the oracle (-m "not gpu"): metrics, free stream, conservation, the survey's
independent cross-check values, brute force at single points, multi-block / permutation equivalence,
boundary-condition fixed points.  SURVEY.md §4 pins 4, 5, 7, 8 and Appendix A."""
import json
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
NG = 6


def make(po, case, threads=None):
    o = po.Oracle(case.dims, case.faces, case.params, threads=threads)
    o.load_case(case)
    return o


# ------------------------------------------------------------------------------------------------
# S1 metrics
# ------------------------------------------------------------------------------------------------
def test_metrics_cartesian_stretched(po, W):
    """Uniform Cartesian grid with spacings (hx,hy,hz): xihat_x = hy hz, etahat_y = hz hx, zetahat_z = hx hy,
    off-diagonals 0, J = 1/(hx hy hz) (Eqs. 7–8 evaluated by hand)."""
    n = (8, 10, 12)
    L = (4.0, 2.5, 24.0)
    X, Y, Z = W._uniform_nodes(n, L)
    xyz = np.stack([X, Y, Z])
    q0 = W.prim_to_cons(1.0 + 0 * X, 0.1 + 0 * X, 0 * X, 0 * X, 1 / 1.4 + 0 * X)
    case = W.Case("cart", [n], [xyz], [q0], W.periodic_faces(0, L), W.default_params(), dt=0.0, steps=0)
    o = make(po, case)
    hx, hy, hz = L[0] / n[0], L[1] / n[1], L[2] / n[2]
    kh = o.field(0, "khat")[:, 3:-3, 3:-3, 3:-3].reshape(3, 3, *[m + 6 for m in n[::-1]])
    jac = o.field(0, "jac")[0, 3:-3, 3:-3, 3:-3]
    ref = np.diag([hy * hz, hz * hx, hx * hy])
    for d in range(3):
        for c in range(3):
            assert np.abs(kh[d, c] - ref[d, c]).max() < 1e-13, (d, c)
    assert np.abs(jac * (hx * hy * hz) - 1).max() < 1e-13


def test_metrics_converge_to_analytic_sixth_order(po, W):
    """J of the C1 mapping vs the analytic Jacobian determinant: error ratio ~ 2^6 per halving."""
    errs = []
    for n in (16, 32):
        case = W.c1_vortex(n)
        o = make(po, case)
        h = 10.0 / n
        X, Y, Z = W._uniform_nodes((n, n, n), (10.0,) * 3)
        s = lambda a: np.sin(np.pi * a / 5)
        c = lambda a: np.pi / 5 * np.cos(np.pi * a / 5)
        # d(x,y,z)/d(X,Y,Z) of x = X + .1 s(Y) s(Z), y = Y + .1 s(Z) s(X), z = Z + .1 s(X) s(Y)
        A = np.array([[1 + 0 * X, .1 * c(Y) * s(Z), .1 * s(Y) * c(Z)],
                      [.1 * s(Z) * c(X), 1 + 0 * X, .1 * c(Z) * s(X)],
                      [.1 * c(X) * s(Y), .1 * s(X) * c(Y), 1 + 0 * X]])
        det = np.linalg.det(np.moveaxis(A, (0, 1), (-2, -1)))
        Jref = 1.0 / (det * h ** 3)
        errs.append(np.abs(o.interior(0, "jac")[0] / Jref - 1).max())
    assert np.log2(errs[0] / errs[1]) > 5.5, errs


def test_metric_identity_discrete(po, W):
    """sum_d delta_d khat^d_c = 0 discretely (what the conservative form Eq. 7 is for)."""
    case = W.c2_freestream(16, viscous=0)
    o = make(po, case)
    kh = o.field(0, "khat").reshape(3, 3, *o.field(0, "jac").shape[1:])
    n = 16
    tot = np.zeros((3, n, n, n))
    for d, ax in ((0, 3), (1, 2), (2, 1)):  # xi -> last array axis
        for c in range(3):
            a = kh[d, c]
            for m, cf in ((1, 0.75), (2, -0.15), (3, 1 / 60)):
                sl_p = [slice(NG, NG + n)] * 3
                sl_m = [slice(NG, NG + n)] * 3
                sl_p[ax - 1] = slice(NG + m, NG + n + m)
                sl_m[ax - 1] = slice(NG - m, NG + n - m)
                tot[c] += cf * (a[tuple(sl_p)] - a[tuple(sl_m)])
    assert np.abs(tot).max() < 1e-14 * np.abs(kh).max() * 50


# ------------------------------------------------------------------------------------------------
# pin 4: free-stream preservation on a wavy grid
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("viscous", [0, 1])
def test_free_stream_preserved_to_roundoff(po, W, viscous):
    case = W.c2_freestream(20, viscous=viscous, amp=0.6)  # 3x the config-2 amplitude: strongly warped
    o = make(po, case)
    J = o.interior(0, "jac")[0]
    assert J.max() / J.min() > 1.5  # the grid really is warped
    o.rhs()
    R = o.interior(0, "r")
    # scale of the summands: J * |khat| * |F| ~ J * h^2 * O(1)
    scale = J.max() * np.abs(o.field(0, "khat")).max() * 3.0
    assert np.abs(R).max() < 1e-13 * scale
    q0 = o.interior(0, "q").copy()
    dt = o.cfl_dt(0.5)
    for _ in range(5):
        o.step(dt)
    assert np.abs(o.interior(0, "q") - q0).max() < 1e-13


# ------------------------------------------------------------------------------------------------
# pin 5: discrete conservation in a periodic domain
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("which", ["vortex-euler", "tgv-ns"])
def test_discrete_conservation(po, W, which):
    case = W.c1_vortex(16) if which == "vortex-euler" else W.tgv_sine_box(16, viscous=1)
    o = make(po, case)
    o.rhs()
    R, J = o.interior(0, "r"), o.interior(0, "jac")[0]
    tot = (R / J).sum(axis=(1, 2, 3))
    mag = np.abs(R / J).sum(axis=(1, 2, 3)) + 1e-30
    assert np.all(np.abs(tot) < 1e-13 * np.maximum(mag, np.abs(R / J).max() * 10)), tot


# ------------------------------------------------------------------------------------------------
# survey Appendix A cross-check values (independent numpy prototype at survey time)
# ------------------------------------------------------------------------------------------------
def test_survey_appendix_a1_euler_vortex(po, W):
    G = json.load(open(os.path.join(HERE, "golden", "survey_appendix_a.json")))["A1"]
    o = make(po, W.c1_vortex(32))
    o.rhs()
    R, J, kh = o.interior(0, "r"), o.interior(0, "jac")[0], o.interior(0, "khat")
    mx = np.abs(R).max(axis=(1, 2, 3))
    assert np.allclose(mx, G["max_abs_R"], rtol=1e-10)
    for pt in G["points"]:
        i, j, k = pt["ijk"]
        assert J[k, j, i] == pytest.approx(pt["J"], rel=1e-13)
        assert np.allclose(R[:, k, j, i], pt["R"], rtol=0, atol=1e-10 * mx.max() * 1e-2), pt
    assert np.allclose(kh[0:3, 11, 7, 5], G["khat_xi_at_5_7_11"], rtol=1e-12)


def test_survey_appendix_a2_viscous_tgv(po, W):
    G = json.load(open(os.path.join(HERE, "golden", "survey_appendix_a.json")))["A2"]
    r = {}
    for v in (0, 1):
        o = make(po, W.tgv_sine_box(16, viscous=v))
        o.rhs()
        r[v] = o.interior(0, "r").copy()
        J = o.interior(0, "jac")[0].copy()
    for pt in G["points"]:
        i, j, k = pt["ijk"]
        assert J[k, j, i] == pytest.approx(pt["J"], rel=1e-13)
        assert np.allclose(r[0][:, k, j, i], pt["R_euler"], rtol=0, atol=2e-14)
        assert np.allclose((r[1] - r[0])[1:, k, j, i], pt["R_visc"], rtol=0, atol=2e-16)


# ------------------------------------------------------------------------------------------------
# pin 8: brute force — the definition evaluated point by point with periodic wrap (no ghost arrays,
# no line buffers), built only from the per-point routines that test_oracle_pointwise.py pins.
# ------------------------------------------------------------------------------------------------
def _brute_rhs_point(po, q, kh, jac, p, params):
    """q: (5,n,n,n) [k,j,i]; kh: (3,3,n,n,n); periodic.  Returns R(5) at p=(i,j,k)."""
    n = q.shape[1:]
    g = params["gamma"]

    def at(arr, idx):  # idx = (i,j,k) with wrap
        return arr[..., idx[2] % n[0], idx[1] % n[1], idx[0] % n[2]]

    def shifted(idx, d, s):
        t = list(idx)
        t[d] += s
        return tuple(t)

    def Fplus_at(idx, d):  # F+ at idx+1/2 from the stencil centred on idx
        k0 = at(kh[d], idx)
        L, R = po.eig(at(q, idx), k0 / np.linalg.norm(k0), g)
        V = np.array([L @ at(q, shifted(idx, d, s)) for s in range(-2, 3)])
        vL = np.array([po.weno5(V[:, f].copy(), params["weno_eps"])[0] for f in range(5)])
        kk = np.array([po.khat_half(np.array([at(kh[d], shifted(idx, d, s))[c] for s in range(-2, 4)])) for c in range(3)])
        return po.sw_flux(R @ vL, kk, +1, g)

    def Fminus_at(idx, d):  # F- at idx-1/2 from the stencil centred on idx
        k0 = at(kh[d], idx)
        L, R = po.eig(at(q, idx), k0 / np.linalg.norm(k0), g)
        V = np.array([L @ at(q, shifted(idx, d, s)) for s in range(-2, 3)])
        vR = np.array([po.weno5(V[:, f].copy(), params["weno_eps"])[1] for f in range(5)])
        kk = np.array([po.khat_half(np.array([at(kh[d], shifted(idx, d, s))[c] for s in range(-3, 3)])) for c in range(3)])
        return po.sw_flux(R @ vR, kk, -1, g)

    def phi(idx):
        Q = at(q, idx)
        u = Q[1:4] / Q[0]
        pr = (g - 1) * (Q[4] - 0.5 * Q[0] * u @ u)
        return np.array([u[0], u[1], u[2], g * pr / Q[0]])

    def grad(idx):
        dphi = np.array([[po.d6(np.array([phi(shifted(idx, d, s))[f] for s in range(-3, 4)])) for f in range(4)] for d in range(3)])
        return po.grad_point(dphi, np.array([at(kh[d], idx) for d in range(3)]), float(at(jac, idx)))

    def Fv(idx, d):
        mu = params["mach"] / params["reynolds"]
        kappa = mu / (params["prandtl"] * (g - 1))
        return po.visc_flux_point(phi(idx)[:3], grad(idx), at(kh[d], idx), mu, kappa)

    accD, accV = np.zeros(5), np.zeros(5)
    for d in range(3):
        fph = Fplus_at(p, d) + Fminus_at(shifted(p, d, 1), d)
        fmh = Fplus_at(shifted(p, d, -1), d) + Fminus_at(p, d)
        F = {s: po.point_flux(at(q, shifted(p, d, s)), at(kh[d], shifted(p, d, s)), g) for s in range(-3, 4)}
        accD += (fph - fmh) + 17 / 256 * (F[1] - F[-1]) - 13 / 320 * (F[2] - F[-2]) + 19 / 3840 * (F[3] - F[-3])
    if params["viscous"]:
        for d in range(3):
            fv = np.array([Fv(shifted(p, d, s), d) for s in range(-3, 4)])
            accV += np.array([po.d6(fv[:, m].copy()) for m in range(5)])
    return float(at(jac, p)) * (accV - accD)


@pytest.mark.parametrize("viscous", [0, 1])
def test_brute_force_single_points(po, W, viscous):
    case = W.tgv_sine_box(12, viscous=viscous, mach=0.4)
    o = make(po, case)
    o.rhs()
    q = o.interior(0, "q").copy()
    kh = o.interior(0, "khat").reshape(3, 3, 12, 12, 12).copy()
    jac = o.interior(0, "jac")[0].copy()
    R = o.interior(0, "r")
    for p in [(0, 0, 0), (11, 5, 2), (3, 11, 7), (6, 6, 11), (1, 10, 0)]:
        ref = _brute_rhs_point(po, q, kh, jac, p, case.params)
        got = R[:, p[2], p[1], p[0]]
        assert np.allclose(got, ref, rtol=0, atol=1e-13 * np.abs(R).max() + 1e-16), (p, got, ref)


# ------------------------------------------------------------------------------------------------
# pin 7: decomposition and permutation equivalence (ghost fill S6 through signed permutations)
# ------------------------------------------------------------------------------------------------
def _multiblock_case(W, G=16, permute=True, seed=5, viscous=1):
    L = 2 * np.pi
    xyz_g, h, _ = W.wavy_box(G, seed, L)
    q_g = W.tgv_field(xyz_g, 0.3)
    rng = np.random.default_rng(seed)
    rots = W.proper_rotations()
    rotations = [rots[int(rng.integers(0, 24))] for _ in range(8)] if permute else None
    dims, xyz, q0, faces, info = W.split_periodic(xyz_g, q_g, (L, L, L), (2, 2, 2), rotations)
    prm = W.default_params(viscous=viscous, mach=0.3, reynolds=200.0)
    single = W.Case("single", [(G, G, G)], [xyz_g], [q_g], W.periodic_faces(0, (L, L, L)), prm, dt=0.0, steps=0)
    multi = W.Case("multi", dims, xyz, q0, faces, prm, dt=0.0, steps=0, meta=dict(info=info, G=(G, G, G)))
    return single, multi


def test_multiblock_identity_rotation_is_bit_identical(po, W):
    single, multi = _multiblock_case(W, permute=False)
    o1, o8 = make(po, single), make(po, multi)
    dt = o1.cfl_dt(0.5)
    for _ in range(2):
        r1 = o1.step(dt)
        r8 = o8.step(dt)
    got = W.gather_blocks([o8.interior(b, "q") for b in range(8)], multi.meta["info"], multi.meta["G"])
    assert np.array_equal(got, o1.interior(0, "q"))
    assert np.allclose(r1, r8, rtol=1e-13)
    # ghost cells of a block equal the neighbour interior (check one whole ghosted array against the wrapped global)
    jac8 = W.gather_blocks([o8.interior(b, "jac") for b in range(8)], multi.meta["info"], multi.meta["G"])
    assert np.array_equal(jac8, o1.interior(0, "jac"))


def test_multiblock_signed_permutations_match_single_block(po, W):
    single, multi = _multiblock_case(W, permute=True)
    assert any(f["perm"] != [0, 1, 2] or f["sign"] != [1, 1, 1] for f in multi.faces)
    o1, o8 = make(po, single), make(po, multi)
    jac8 = W.gather_blocks([o8.interior(b, "jac") for b in range(8)], multi.meta["info"], multi.meta["G"])
    assert np.allclose(jac8, o1.interior(0, "jac"), rtol=1e-12)
    o1.rhs()
    o8.rhs()
    R1 = o1.interior(0, "r")
    R8 = W.gather_blocks([o8.interior(b, "r") for b in range(8)], multi.meta["info"], multi.meta["G"])
    assert np.abs(R8 - R1).max() < 1e-12 * np.abs(R1).max()
    dt = o1.cfl_dt(0.5)
    for _ in range(3):
        o1.step(dt)
        o8.step(dt)
    got = W.gather_blocks([o8.interior(b, "q") for b in range(8)], multi.meta["info"], multi.meta["G"])
    assert np.abs(got - o1.interior(0, "q")).max() < 1e-12


def test_ghost_fill_edges_and_corners(po, W):
    """After the three-pass fill every ghost cell (faces, edges, corners) of every block holds the periodic
    image of the global field, and ghost coordinates hold the shifted image."""
    single, multi = _multiblock_case(W, permute=True, viscous=0)
    o8 = make(po, multi)
    G = 16
    qg, xg = single.q0[0], single.xyz[0]
    L = 2 * np.pi
    for b, inf in enumerate(multi.meta["info"]):
        n = inf["n"]
        l2, l1, l0 = np.meshgrid(*(np.arange(-NG, n[a] + NG) for a in (2, 1, 0)), indexing="ij")
        loc = [l0, l1, l2]
        gi = [None] * 3
        for a in range(3):
            A = inf["gax"][a]
            r = loc[a] if inf["gsg"][a] > 0 else n[a] - 1 - loc[a]
            gi[A] = inf["origin"][A] + r
        want_q = qg[:, gi[2] % G, gi[1] % G, gi[0] % G]
        assert np.array_equal(o8.field(b, "q"), want_q)
        want_x = xg[:, gi[2] % G, gi[1] % G, gi[0] % G] + np.stack([L * np.floor_divide(gi[A], G) for A in range(3)])
        assert np.allclose(o8.field(b, "xyz"), want_x, rtol=0, atol=1e-13)


# ------------------------------------------------------------------------------------------------
# S5 boundary conditions (readings U13, U14): fixed points and symmetries
# ------------------------------------------------------------------------------------------------
def _small_cylinder(W, mach, noise=0.0, **kw):
    return W.c5_cylinder(ni=32, nj=14, nk=8, ratio=1.25, r_out=8.0, mach=mach, noise=noise, **kw)


def test_cylinder_grid_orientation_and_wall_ghosts(po, W):
    case = _small_cylinder(W, mach=0.2, noise=1e-3)
    o = make(po, case)
    J = o.field(0, "jac")[0, 3:-3, 3:-3, 3:-3]
    assert J.min() > 0
    q = o.field(0, "q")
    # wall nodes: zero momentum; ghosts: even rho/e, odd momentum (tangential range [-3, n+3))
    t = slice(3, -3)
    assert np.all(q[1:4, t, NG, t] == 0.0)
    for g in range(1, NG + 1):
        assert np.array_equal(q[0, t, NG - g, t], q[0, t, NG + g, t])
        assert np.array_equal(q[4, t, NG - g, t], q[4, t, NG + g, t])
        assert np.array_equal(q[1:4, t, NG - g, t], -q[1:4, t, NG + g, t])
    # far-field ghosts copy the boundary node
    for g in range(1, NG + 1):
        assert np.array_equal(q[:, t, -NG - 1 + g, t], q[:, t, -NG - 1, t])
    # wall ghost coordinates are point reflections; outer ghosts are linear extrapolations
    x = o.field(0, "xyz")
    assert np.allclose(x[:, :, NG - 2, :], 2 * x[:, :, NG, :] - x[:, :, NG + 2, :], atol=1e-14)
    assert np.allclose(x[:, :, -NG - 1 + 3, :], x[:, :, -NG - 1, :] + 3 * (x[:, :, -NG - 1, :] - x[:, :, -NG - 2, :]), atol=1e-13)


def test_fluid_at_rest_is_a_fixed_point_with_wall_and_farfield(po, W):
    case = _small_cylinder(W, mach=0.0)
    case.params["mach"] = 0.2  # viscosity scale only; the state itself is at rest
    o = make(po, case)
    q0 = o.interior(0, "q").copy()
    o.rhs()
    J = o.interior(0, "jac")[0]
    assert np.abs(o.interior(0, "r")).max() < 1e-12 * J.max() * np.abs(o.field(0, "khat")[:, 3:-3, 3:-3, 3:-3]).max()
    dt = 0.3 * o.cfl_dt(1.0)
    for _ in range(3):
        o.step(dt)
    assert np.abs(o.interior(0, "q") - q0).max() < 1e-13


def test_uniform_flow_is_a_fixed_point_of_the_farfield_bc(po, W):
    """Block with FARFIELD on both eta faces (periodic otherwise), uniform oblique flow = q_inf."""
    n = (10, 12, 8)
    L = (2.0, 2.4, 1.6)
    X, Y, Z = W._uniform_nodes(n, L)
    xyz = np.stack([X + 0.03 * np.sin(np.pi * Y / 1.2), Y, Z + 0.02 * np.sin(2 * np.pi * X / 2.0)])
    qinf = W.prim_to_cons(1.0, 0.3, 0.25, -0.1, 1 / 1.4)
    q0 = np.broadcast_to(qinf[:, None, None, None], (5, n[2], n[1], n[0])).copy()
    faces = [f for f in W.periodic_faces(0, L) if f["face"] not in (2, 3)]
    for s in (2, 3):
        faces.append(dict(block=0, face=s, type=W.FARFIELD, nbr_block=-1, nbr_face=-1, perm=[0, 1, 2], sign=[1, 1, 1], shift=[0.0] * 3))
    case = W.Case("ff", [n], [xyz], [q0], faces, W.default_params(viscous=1, mach=0.4, q_inf=qinf), dt=0.0, steps=0)
    o = make(po, case)
    dt = o.cfl_dt(0.5)
    for _ in range(3):
        o.step(dt)
    assert np.abs(o.interior(0, "q") - q0).max() < 2e-13


def test_farfield_supersonic_branches(po, W):
    """Supersonic outflow copies the interior neighbour; supersonic inflow imposes q_inf."""
    n = (8, 8, 8)
    L = (1.0, 1.0, 1.0)
    X, Y, Z = W._uniform_nodes(n, L)
    xyz = np.stack([X, Y, Z])
    qinf = W.prim_to_cons(1.0, 0.0, 2.0, 0.0, 1 / 1.4)  # Mach 2 along +y: face 2 (-eta) inflow, face 3 (+eta) outflow
    rng = np.random.default_rng(3)
    q0 = W.prim_to_cons(1.0 + 0.05 * rng.random(X.shape), 0.05 * rng.random(X.shape), 2.0 + 0.05 * rng.random(X.shape),
                        0 * X, 1 / 1.4 + 0.02 * rng.random(X.shape))
    faces = [f for f in W.periodic_faces(0, L) if f["face"] not in (2, 3)]
    for s in (2, 3):
        faces.append(dict(block=0, face=s, type=W.FARFIELD, nbr_block=-1, nbr_face=-1, perm=[0, 1, 2], sign=[1, 1, 1], shift=[0.0] * 3))
    case = W.Case("ffs", [n], [xyz], [q0], faces, W.default_params(viscous=0, mach=2.0, q_inf=qinf), dt=0.0, steps=0)
    o = make(po, case)
    q = o.field(0, "q")
    t = slice(NG, -NG)
    assert np.allclose(q[:, t, NG, t], qinf[:, None, None], rtol=1e-14)            # inflow plane j = 0
    assert np.allclose(q[:, t, -NG - 1, t], q[:, t, -NG - 2, t], rtol=1e-14)       # outflow plane j = n-1 <- j = n-2


def test_create_rejects_bad_topology(po, W):
    case = W.c1_vortex(8)
    bad = [dict(f) for f in case.faces]
    bad[0]["sign"] = [-1, 1, 1]  # improper rotation
    with pytest.raises(ValueError):
        po.Oracle(case.dims, bad, case.params)
    bad = [dict(f) for f in case.faces]
    bad[0]["nbr_face"] = 3  # axis mismatch with perm
    with pytest.raises(ValueError):
        po.Oracle(case.dims, bad, case.params)


# ------------------------------------------------------------------------------------------------
# Physical boundary conditions NEXT to block interfaces (Fig. 2's bc_block -> bc_phys order; U12-U15):
# the cylinder cut along the azimuth into point-matched blocks must reproduce the single-block cylinder.
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("nblk", [2, 3])
def test_split_cylinder_with_wall_and_far_field_matches_single_block(po, W, nblk):
    multi = W.c5_cylinder_split(nblk, ni=48, nj=14, nk=8, noise=1e-2)
    single = multi.meta["single"]
    o1, om = make(po, single), make(po, multi)
    nb = multi.dims[0][0]
    cat = lambda name: np.concatenate([om.interior(b, name) for b in range(nblk)], axis=-1)
    # metrics: the ghost coordinates behind an interface are the neighbour's nodes, behind wall / far field the same
    # reflection / extrapolation as in the single block
    assert np.array_equal(cat("jac"), o1.interior(0, "jac"))
    assert np.array_equal(cat("khat"), o1.interior(0, "khat"))
    # R agrees bit for bit on every node the scheme advances.  On the two node planes that the physical BCs own (j = 0 wall,
    # j = nj-1 far field) R is never used -- the BC overwrites those nodes after every stage -- and there it depends on
    # ghost cells outside the range the BC refreshes (the viscous reach is +-6 along xi, the BC covers the tangential range
    # [-3, n+3)): those hold the image of the node plane from BEFORE the BC, whichever block they were copied from.
    o1.rhs()
    om.rhs()
    R1, Rm = o1.interior(0, "r"), cat("r")
    assert np.array_equal(Rm[:, :, 1:-1], R1[:, :, 1:-1])
    assert np.abs(Rm - R1).max() < 1e-3 * np.abs(R1).max()
    dt = o1.cfl_dt(0.5)
    assert om.cfl_dt(0.5) == dt
    for _ in range(4):
        r1 = o1.step(dt)
        rm = om.step(dt)
    assert np.array_equal(cat("q"), o1.interior(0, "q"))
    # U17a: the residual sums R^2 over the INNER points, i.e. without the node planes the physical BCs own, so
    # it no longer sees the stale ghost images those planes read: the cut cylinder reports the single block's residual
    assert np.allclose(r1, rm, rtol=1e-13, atol=0.0)
    # the wall did something: the velocity at the wall nodes is zero, away from it not
    q = cat("q")
    assert np.abs(q[1:4, :, 0, :]).max() == 0.0 and np.abs(q[1, :, 3, :]).max() > 0.05
    assert nb * nblk == 48
