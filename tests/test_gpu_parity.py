"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI, against the CPU oracle element by
element on the same seeded inputs.  Tolerances (BASELINE.json north_star): 1e-12 max relative error per
RHS evaluation, normalised per equation by the magnitude of the summands S_m = max J * max_d |F^d_m|
(SURVEY §8(d) "Parity normaliser"); 1e-10 on the state after 100 RK3 steps (smooth cases); integer /
copy work (ghost fill) bit-exact."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
NG = 6
RHS_TOL = 1e-12


@pytest.fixture(scope="module")
def B():
    import torch

    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2006_07964_b200 import binding

    return binding


def pair(po, B, case):
    o = po.Oracle(case.dims, case.faces, case.params)
    o.load_case(case)
    g = B.Context(case.dims, case.faces, case.params)
    g.load_case(case)
    return o, g


def flux_scale(o, b, gamma=1.4):
    """S_m = max J * max over directions and points of |F^d_m(Q, khat^d)| on the interior (Eq. 4)."""
    q = o.interior(b, "q")
    kh = o.interior(b, "khat").reshape(3, 3, *q.shape[1:])
    J = o.interior(b, "jac")[0]
    u = q[1:4] / q[0]
    p = (gamma - 1) * (q[4] - 0.5 * q[0] * (u ** 2).sum(0))
    S = np.zeros(5)
    for d in range(3):
        th = (kh[d] * u).sum(0)
        F = np.stack([q[0] * th, q[1] * th + kh[d, 0] * p, q[2] * th + kh[d, 1] * p, q[3] * th + kh[d, 2] * p, (q[4] + p) * th])
        S = np.maximum(S, np.abs(F).max(axis=(1, 2, 3)))
    return S * J.max()


def assert_rhs_parity(o, g, case, tol=RHS_TOL):
    o.rhs()
    g.rhs()
    worst = 0.0
    for b in range(len(case.dims)):
        S = flux_scale(o, b)
        ro, rg = o.interior(b, "r"), g.to_numpy(b, "r")
        assert np.isfinite(rg).all()
        err = np.abs(rg - ro).max(axis=(1, 2, 3)) / S
        worst = max(worst, err.max())
        assert err.max() < tol, (case.name, b, err)
    return worst


# ------------------------------------------------------------------------------------------------
# S1 metrics
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("which", ["c1", "wavy-ragged", "cylinder", "multiblock"])
def test_metrics_parity(po, W, B, which):
    case = {"c1": lambda: W.c1_vortex(32),
            "wavy-ragged": lambda: ragged_case(W),
            "cylinder": lambda: W.c5_cylinder(ni=64, nj=24, nk=10, ratio=1.15, r_out=10.0),
            "multiblock": lambda: W.c4_multiblock(nb=12)}[which]()
    o, g = pair(po, B, case)
    for b in range(len(case.dims)):
        xo, xg = o.field(b, "xyz"), g.to_numpy(b, "xyz", interior=False)
        assert np.allclose(xg, xo, rtol=0, atol=1e-13 * np.abs(xo).max())
        box = (slice(None),) + (slice(3, -3),) * 3
        ko, kg = o.field(b, "khat")[box], g.to_numpy(b, "khat", interior=False)[box]
        assert np.abs(kg - ko).max() < 1e-13 * np.abs(ko).max()
        jo, jg = o.field(b, "jac")[box], g.to_numpy(b, "jac", interior=False)[box]
        assert np.abs(jg / jo - 1).max() < 1e-12


def ragged_case(W, viscous=1, n=(71, 23, 15)):
    """Non-cubic block whose sizes are not multiples of any tile edge (62, 6, 32): several tiles + ragged tails.
    ni odd: the xi sweep cannot use TMA (row pitch not a multiple of 16 bytes) and runs the cp.async kernel;
    n = (70, 45, 9): TMA xi sweep with ni % 4 = 2, a partial 32-line group and several segments."""
    L = 2 * np.pi
    X, Y, Z = W._uniform_nodes(n, (L, L, L))
    modes = W.wavy_modes(11)
    xyz = W.wavy_mapping(X, Y, Z, L, L / 23, modes, amp=0.25)
    q0 = W.tgv_field(xyz, 0.4)
    q0 = W.prim_to_cons(q0[0] * (1 + 0.1 * np.sin(xyz[1])), q0[1] / q0[0] + 0.2, q0[2] / q0[0], 0.1 * np.cos(xyz[0] + xyz[2]),
                        (1 / 1.4) * (1 + 0.05 * np.cos(xyz[2])))
    return W.Case("ragged", [n], [xyz], [q0], W.periodic_faces(0, (L, L, L)),
                  W.default_params(viscous=viscous, mach=0.4, reynolds=300.0), dt=1e-3, steps=0)


def test_fastmath_accuracy(B):
    """csrc/fastmath.cuh (MUFU seed + one cubic Newton step) against correctly rounded 1/x and 1/sqrt(x) over the
    magnitudes the kernels feed it (rho, c^2, |khat|^2 ~ 1e-6..1e6; WENO denominators down to (4 eps)^8 ~ 1e-43)."""
    rng = np.random.default_rng(5)
    x = np.concatenate([rng.uniform(0.5, 2.0, 20000), 10.0 ** rng.uniform(-45, 40, 20000), [1.0, 2.0, 4.0, 0.25, 3.0]])
    r, s = B.selftest_fastmath(x)
    exact_r = (1.0 / x.astype(np.longdouble))
    exact_s = 1.0 / np.sqrt(x.astype(np.longdouble))
    er = np.abs((r - exact_r) / exact_r).max()
    es = np.abs((s - exact_s) / exact_s).max()
    assert er < 4.5e-16 and es < 4.5e-16, (float(er), float(es))  # <= 2 ulp


# ------------------------------------------------------------------------------------------------
# S2 + S3: RHS parity, element by element
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("which", ["c1-euler", "tgv-ns", "ragged-ns", "ragged-euler", "ragged-even-ns", "ragged-even-euler",
                                   "multiblock-ns", "cylinder-ns", "tiny"])
def test_rhs_parity(po, W, B, which):
    case = {"c1-euler": lambda: W.c1_vortex(32),
            "ragged-even-ns": lambda: ragged_case(W, 1, n=(70, 45, 9)),
            "ragged-even-euler": lambda: ragged_case(W, 0, n=(70, 45, 9)),
            "tgv-ns": lambda: W.tgv_sine_box(24, viscous=1, mach=0.4),
            "ragged-ns": lambda: ragged_case(W, 1),
            "ragged-euler": lambda: ragged_case(W, 0),
            "multiblock-ns": lambda: W.c4_multiblock(nb=12, mach=0.3),
            "cylinder-ns": lambda: W.c5_cylinder(ni=64, nj=24, nk=10, ratio=1.15, r_out=10.0, noise=1e-2),
            "tiny": lambda: W.tgv_sine_box(6, viscous=1, mach=0.3)}[which]()  # minimum block size (degenerate tiles)
    o, g = pair(po, B, case)
    assert_rhs_parity(o, g, case)


@pytest.mark.parametrize("plan", [4, 5])
@pytest.mark.parametrize("which", ["ragged-ns", "ragged-euler", "ragged-even-ns", "multiblock-ns", "cylinder-ns", "tiny"])
def test_rhs_parity_other_sweep_plans(po, W, B, which, plan):
    """cfd_set_sweep_plan: the xi sweep with the 8-byte cp.async staging kernel forced (4) and with the TMA-fed chunk
    ring (5) against the oracle (plan 0, the 16-byte cp.async chunk ring, is the default everywhere else)."""
    case = {"ragged-ns": lambda: ragged_case(W, 1),
            "ragged-euler": lambda: ragged_case(W, 0),
            "ragged-even-ns": lambda: ragged_case(W, 1, n=(70, 45, 9)),
            "multiblock-ns": lambda: W.c4_multiblock(nb=12, mach=0.3),
            "cylinder-ns": lambda: W.c5_cylinder(ni=64, nj=24, nk=10, ratio=1.15, r_out=10.0, noise=1e-2),
            "tiny": lambda: W.tgv_sine_box(6, viscous=1, mach=0.3)}[which]()
    o, g = pair(po, B, case)
    g.set_sweep_plan(plan)
    assert_rhs_parity(o, g, case)


# NEXT-1: the original AFWENO ordering (scheme = 1, Fig. 9, reading U7) on the CUDA path against the oracle's
# scheme 1 (pinned by tests/test_oracle_order.py: fifth order on a smooth line, exactness, free stream)
@pytest.mark.parametrize("which", ["c1-euler", "tgv-ns", "ragged-ns", "ragged-euler", "ragged-even-ns", "ragged-even-euler",
                                   "multiblock-ns", "cylinder-ns", "tiny", "strong-gradients"])
def test_rhs_parity_scheme1_original_afweno(po, W, B, which):
    case = {"c1-euler": lambda: W.c1_vortex(32),
            "ragged-even-ns": lambda: ragged_case(W, 1, n=(70, 45, 9)),
            "ragged-even-euler": lambda: ragged_case(W, 0, n=(70, 45, 9)),
            "tgv-ns": lambda: W.tgv_sine_box(24, viscous=1, mach=0.4),
            "ragged-ns": lambda: ragged_case(W, 1),
            "ragged-euler": lambda: ragged_case(W, 0),
            "multiblock-ns": lambda: W.c4_multiblock(nb=12, mach=0.3),
            "cylinder-ns": lambda: W.c5_cylinder(ni=64, nj=24, nk=10, ratio=1.15, r_out=10.0, noise=1e-2),
            "tiny": lambda: W.tgv_sine_box(6, viscous=1, mach=0.3),
            "strong-gradients": lambda: noisy_vortex_case(W)}[which]()
    case.params["scheme"] = 1
    o, g = pair(po, B, case)
    assert_rhs_parity(o, g, case)
    # the two schemes are different discretisations: the comparison above is not vacuous
    if which == "strong-gradients":
        case.params["scheme"] = 0
        o0 = po.Oracle(case.dims, case.faces, case.params)
        o0.load_case(case)
        o0.rhs()
        assert np.abs(o0.interior(0, "r") - o.interior(0, "r")).max() > 1e-6 * np.abs(o.interior(0, "r")).max()


def test_scheme1_fused_steps_match_oracle(po, W, B):
    """Three RK3 steps with cfd_stage_fused under scheme 1 (ragged viscous block, several tiles and segments)."""
    case = ragged_case(W, 1, n=(70, 45, 9))
    case.params["scheme"] = 1
    o, g = pair(po, B, case)
    dt = o.cfl_dt(0.5)
    for _ in range(3):
        ro = o.step(dt)
        rg = g.step(dt, want_res=True)
    assert np.allclose(rg, ro, rtol=1e-10)
    qo, qg = o.interior(0, "q"), g.to_numpy(0, "q")
    assert np.abs(qg - qo).max() < 1e-12 * np.abs(qo).max()
    with pytest.raises(B.CfdError):  # plans 1-3 and 6 (tiled kernels) were retired in round 2
        g.set_sweep_plan(1)


def noisy_vortex_case(W):
    """Non-smooth data (the WENO weights far from the linear ones): seeded random +-20 % perturbation per node."""
    case = W.c1_vortex(24)
    rng = np.random.default_rng(99)
    q = case.q0[0]
    rho = q[0] * (1 + 0.2 * rng.uniform(-1, 1, q[0].shape))
    p = (1 / 1.4) * (1 + 0.2 * rng.uniform(-1, 1, q[0].shape))
    case.q0[0] = W.prim_to_cons(rho, q[1] / q[0], q[2] / q[0] + 0.3 * rng.uniform(-1, 1, q[0].shape), q[3] / q[0], p)
    return case


def test_rhs_parity_strong_gradients(po, W, B):
    o, g = pair(po, B, noisy_vortex_case(W))
    assert_rhs_parity(o, g, noisy_vortex_case(W))


def test_free_stream_on_gpu(po, W, B):
    """Config 2 (reduced to 32^3): uniform flow on the seeded wavy grid stays at round-off on the GPU itself."""
    case = W.c2_freestream(32, viscous=1)
    g = B.Context(case.dims, case.faces, case.params)
    g.load_case(case)
    g.rhs()
    r = g.to_numpy(0, "r")
    J = g.to_numpy(0, "jac")
    kh = g.to_numpy(0, "khat")
    assert np.abs(r).max() < 1e-12 * J.max() * np.abs(kh).max() * 3
    q0 = g.to_numpy(0, "q").copy()
    for _ in range(100):
        g.step(case.dt)
    assert np.abs(g.to_numpy(0, "q") - q0).max() < 1e-12


# ------------------------------------------------------------------------------------------------
# S6 / S5: ghost fill (bit-exact) and boundary conditions
# ------------------------------------------------------------------------------------------------
def test_exchange_is_bit_exact_with_signed_permutations(po, W, B):
    case = W.c4_multiblock(nb=10, mach=0.3)
    assert any(f["perm"] != [0, 1, 2] for f in case.faces)
    o, g = pair(po, B, case)
    for b in range(8):
        assert np.array_equal(g.to_numpy(b, "q", interior=False), o.field(b, "q"))
    # scramble the ghosts on the GPU, exchange again
    for b in range(8):
        f = g.field(b, "q")
        keep = f[:, NG:-NG, NG:-NG, NG:-NG].clone()
        f.fill_(float("nan"))
        f[:, NG:-NG, NG:-NG, NG:-NG] = keep
    g.exchange_interfaces()
    for b in range(8):
        assert np.array_equal(g.to_numpy(b, "q", interior=False), o.field(b, "q"))


def test_bc_parity_cylinder(po, W, B):
    case = W.c5_cylinder(ni=48, nj=20, nk=8, ratio=1.2, r_out=8.0, noise=1e-2)
    o, g = pair(po, B, case)
    qo, qg = o.field(0, "q"), g.to_numpy(0, "q", interior=False)
    t = slice(3, -3)  # tangential range the BCs define
    assert np.allclose(qg[:, t, :, t], qo[:, t, :, t], rtol=1e-13, atol=1e-15)
    assert np.all(qg[1:4, t, NG, t] == 0.0)


# ------------------------------------------------------------------------------------------------
# S4 and whole steps
# ------------------------------------------------------------------------------------------------
def test_rk_stage_residual_leaves_out_bc_owned_node_planes(po, W, B):
    """U17a on both S4 kernels (k_rk<1> of cfd_rk_stage, the fused zeta sweep of cfd_stage_fused): cylinder block with WALL
    and FARFIELD faces; the residual equals the oracle's (which is pinned to the sum over j = 1 .. nj-2 of its own R field)."""
    case = W.c5_cylinder(ni=64, nj=24, nk=10, ratio=1.15, r_out=10.0, noise=1e-2)
    o, g = pair(po, B, case)
    o.rhs()
    g.rhs()
    R = g.to_numpy(0, "r").astype(np.longdouble)
    inner = (R[:, :, 1:-1, :] ** 2).sum(axis=(1, 2, 3)).astype(float)
    ro = o.rk_stage(1, 1e-3, want_res=True)
    rg = g.rk_stage(1, 1e-3, want_res=True)
    assert np.allclose(rg, ro, rtol=1e-12, atol=0.0)
    assert np.allclose(rg, inner, rtol=1e-12, atol=0.0)
    o2, g2 = pair(po, B, case)
    assert np.allclose(g2.stage_fused(1, 1e-3, want_res=True), o2.stage(1, 1e-3, want_res=True), rtol=1e-12, atol=0.0)


def test_rk_stage_and_residual(po, W, B):
    case = ragged_case(W, 1)
    o, g = pair(po, B, case)
    o.rhs()
    g.rhs()
    dt = 1e-3
    for s in (1, 2, 3):
        ro = o.rk_stage(s, dt, want_res=True)
        rg = g.rk_stage(s, dt, want_res=True)
        if s == 1:
            assert np.allclose(rg, ro, rtol=1e-12)
        assert np.abs(g.to_numpy(0, "q") - o.interior(0, "q")).max() < 1e-13
    assert np.abs(g.to_numpy(0, "qn") - o.interior(0, "qn")).max() < 1e-13
    # deterministic reduction: bit-identical on repetition
    g.rhs()
    a = g.rk_stage(1, 0.0, want_res=True)
    g.rhs()
    b = g.rk_stage(1, 0.0, want_res=True)
    assert np.array_equal(a, b)


@pytest.mark.parametrize("which", ["c1", "multiblock", "cylinder"])
def test_state_parity_after_steps(po, W, B, which):
    case, nsteps = {"c1": lambda: (W.c1_vortex(32), 10),  # config 1 as specified: 10 RK3 steps at CFL 0.5
                    "multiblock": lambda: (W.c4_multiblock(nb=12, mach=0.3), 6),
                    "cylinder": lambda: (W.c5_cylinder(ni=48, nj=20, nk=8, ratio=1.2, r_out=8.0, noise=1e-3), 6)}[which]()
    o, g = pair(po, B, case)
    dt = o.cfl_dt(0.5)
    for _ in range(nsteps):
        ro = o.step(dt)
        rg = g.step(dt, want_res=True)
    assert np.allclose(rg, ro, rtol=1e-9)
    for b in range(len(case.dims)):
        qo, qg = o.interior(b, "q"), g.to_numpy(b, "q")
        assert np.abs(qg - qo).max() < 1e-11 * np.abs(qo).max()
    if which == "c1":
        exact = W.vortex_field(case.xyz[0], t=nsteps * dt)
        assert np.abs(g.to_numpy(0, "q") - exact).max() < 0.05


@pytest.mark.parametrize("which", ["ragged-ns", "ragged-euler", "multiblock"])
def test_fused_stage_matches_unfused_and_oracle(po, W, B, which):
    """cfd_stage_fused (RK update inside the zeta sweep, buffer roles exchanged, R never stored) against cfd_stage
    (four separate calls) and the oracle: state after 2 steps, q^n after stage 1, the stage-1 residual, and the
    bookkeeping of cfd_buffer_roles."""
    case = {"ragged-ns": lambda: ragged_case(W, 1), "ragged-euler": lambda: ragged_case(W, 0),
            "multiblock": lambda: W.c4_multiblock(nb=10, mach=0.3)}[which]()
    o, g = pair(po, B, case)
    g2 = B.Context(case.dims, case.faces, case.params)
    g2.load_case(case)
    dt = o.cfl_dt(0.5)
    assert g.buffer_roles() == (0, 1, 2)
    ro = o.stage(1, dt, want_res=True)
    rg = g.stage_fused(1, dt, want_res=True)
    r2 = g2.stage(1, dt, want_res=True)
    assert g.buffer_roles() == (2, 0, 1) and g2.buffer_roles() == (0, 1, 2)
    assert np.allclose(rg, r2, rtol=1e-12)
    assert np.allclose(rg, ro, rtol=1e-11)
    for b in range(len(case.dims)):
        assert np.array_equal(g.to_numpy(b, "qn"), g2.to_numpy(b, "qn"))  # the old q buffer, untouched
        assert np.abs(g.to_numpy(b, "q") - g2.to_numpy(b, "q")).max() < 1e-13
        assert np.abs(g.to_numpy(b, "q") - o.interior(b, "q")).max() < 1e-13 * max(1.0, np.abs(o.interior(b, "q")).max())
    for s in (2, 3):
        g.stage_fused(s, dt)
        g2.stage(s, dt)
    assert g.buffer_roles() == (2, 0, 1)
    g.step(dt)
    g2.step(dt, fused=False)
    assert sorted(g.buffer_roles()) == [0, 1, 2]
    for b in range(len(case.dims)):
        a, c = g.to_numpy(b, "q"), g2.to_numpy(b, "q")
        assert np.abs(a - c).max() < 1e-12 * np.abs(c).max()

    # bit-identical on repetition (fixed-order residual, no atomics)
    g3 = B.Context(case.dims, case.faces, case.params)
    g3.load_case(case)
    assert np.array_equal(g3.stage_fused(1, dt, want_res=True), rg)


def test_state_parity_after_100_steps_smooth(po, W, B):
    """north_star: 1e-10 after 100 RK3 steps on smooth cases (TGV, viscous, wavy grid; reduced to 24^3)."""
    case = W.c3_tgv(n=24, viscous=1, mach=0.1)
    o, g = pair(po, B, case)
    dt = o.cfl_dt(0.5)
    for _ in range(100):
        o.step(dt)
        g.step(dt)
    qo, qg = o.interior(0, "q"), g.to_numpy(0, "q")
    assert np.abs(qg - qo).max() < 1e-10 * np.abs(qo).max()


# ------------------------------------------------------------------------------------------------
# Full-size configs in the launch configuration bench.py times: sampled sub-boxes.  The GPU's own q,
# khat, jac (with ghosts) are cut out around sample points and handed to the oracle as a face-less block;
# the oracle's RHS on the sub-box interior must match the GPU's RHS there.
# ------------------------------------------------------------------------------------------------
def subbox_check(po, g, case, b, lo, ext, S):
    sl = tuple(slice(lo[a], lo[a] + ext[a] + 2 * NG) for a in (2, 1, 0))  # array coordinates (ghost offset included)
    o = po.Oracle([tuple(ext)], [], case.params)
    for name in ("q", "khat", "jac"):
        o.field(0, name)[...] = g.field(b, name)[(slice(None),) + sl].cpu().numpy()
    o.rhs()
    isl = tuple(slice(lo[a] + NG, lo[a] + NG + ext[a]) for a in (2, 1, 0))
    rg = g.field(b, "r")[(slice(None),) + isl].cpu().numpy()
    err = np.abs(rg - o.interior(0, "r")).max(axis=(1, 2, 3)) / S
    assert err.max() < RHS_TOL, (case.name, b, lo, err)


def sample_boxes(n, rng, ext=(14, 10, 8), count=5):
    boxes = [(0, 0, 0), tuple(n[a] - ext[a] for a in range(3))]  # the two extreme corners
    for _ in range(count):
        boxes.append(tuple(int(rng.integers(0, n[a] - ext[a] + 1)) for a in range(3)))
    return boxes, ext


@pytest.mark.parametrize("which", ["C2-64", "C3-128", "C4-8x96", "C5-cylinder", "sweep-256", "C3-128-scheme1", "sweep-256-scheme1"])
def test_full_size_sampled_parity(po, W, B, which):
    import torch

    case = {"C2-64": lambda: W.c2_freestream(64), "C3-128": lambda: W.c3_tgv(128), "C4-8x96": lambda: W.c4_multiblock(96),
            "C5-cylinder": lambda: W.c5_cylinder(), "sweep-256": lambda: W.sweep_block(256)}[which.replace("-scheme1", "")]()
    if which.endswith("scheme1"):
        case.params["scheme"] = 1
    g = B.Context(case.dims, case.faces, case.params)
    g.load_case(case)
    g.step(case.dt)  # one full step first so that the sampled state is not the analytic initial field
    g.rhs()
    torch.cuda.synchronize()
    rng = np.random.default_rng(1234)
    for b in range(len(case.dims)):   # every block (C4: all eight, each with its own signed permutation)
        n = case.dims[b]
        q = g.interior(b, "q")
        assert torch.isfinite(q).all()
        # flux scale from the GPU state (tolerance normaliser only)
        u = (q[1:4] / q[0])
        p = 0.4 * (q[4] - 0.5 * q[0] * (u ** 2).sum(0))
        kh = g.interior(b, "khat").reshape(3, 3, *q.shape[1:])
        J = g.interior(b, "jac")[0]
        S = np.zeros(5)
        for d in range(3):
            th = (kh[d] * u).sum(0)
            F = [q[0] * th, q[1] * th + kh[d, 0] * p, q[2] * th + kh[d, 1] * p, q[3] * th + kh[d, 2] * p, (q[4] + p) * th]
            S = np.maximum(S, np.array([float(f.abs().max()) for f in F]))
        S = S * float(J.max())
        boxes, ext = sample_boxes(n, rng, count=5 if b in (0, len(case.dims) - 1) else 2)
        for lo in boxes:
            subbox_check(po, g, case, b, lo, ext, S)


@pytest.mark.parametrize("which", ["C4-8x96", "sweep-256"])
def test_full_size_fused_stage_sampled(po, W, B, which):
    """cfd_stage_fused at full size, in the launch configuration bench.py times: around sampled points the oracle
    recomputes R from the GPU's own state before the stage (sub-box with its ghosts); the GPU's state after stage 1 must
    equal Q + dt R there (Eq. 20), and Q^n must be the old state bit for bit."""
    import torch

    case = {"C4-8x96": lambda: W.c4_multiblock(96), "sweep-256": lambda: W.sweep_block(256)}[which]()
    g = B.Context(case.dims, case.faces, case.params)
    g.load_case(case)
    g.step(case.dt)
    torch.cuda.synchronize()
    rng = np.random.default_rng(4321)
    b = len(case.dims) - 1
    n = case.dims[b]
    boxes, ext = sample_boxes(n, rng, count=4)
    saved = []
    for lo in boxes:
        sl = tuple(slice(lo[a], lo[a] + ext[a] + 2 * NG) for a in (2, 1, 0))
        saved.append({name: g.field(b, name)[(slice(None),) + sl].cpu().numpy().copy() for name in ("q", "khat", "jac")})
    g.stage_fused(1, case.dt)
    torch.cuda.synchronize()
    for lo, sv in zip(boxes, saved):
        o = po.Oracle([tuple(ext)], [], case.params)
        for name in ("q", "khat", "jac"):
            o.field(0, name)[...] = sv[name]
        o.rhs()
        isl = tuple(slice(lo[a] + NG, lo[a] + NG + ext[a]) for a in (2, 1, 0))
        q_old = o.interior(0, "q")
        expect = q_old + case.dt * o.interior(0, "r")
        got = g.field(b, "q")[(slice(None),) + isl].cpu().numpy()
        qn = g.field(b, "qn")[(slice(None),) + isl].cpu().numpy()
        scale = np.abs(q_old).max()  # the field's max magnitude (w ~ 0 in the TGV field: no per-component scale)
        err = np.abs(got - expect).max(axis=(1, 2, 3)) / scale
        assert err.max() < 1e-12, (which, lo, err)
        assert np.array_equal(qn, q_old)


# ------------------------------------------------------------------------------------------------
# error behaviour through the ABI
# ------------------------------------------------------------------------------------------------
def test_error_codes(W, B):
    case = W.c1_vortex(8)
    g = B.Context(case.dims, case.faces, case.params)
    g.load_case(case)
    with pytest.raises(B.CfdError) as e:
        g.rk_stage(4, 0.1)
    assert e.value.code == -4
    bad = [dict(f) for f in case.faces]
    bad[0]["sign"] = [-1, 1, 1]
    with pytest.raises(B.CfdError) as e:
        B.Context(case.dims, bad, case.params)
    assert e.value.code == -2
    with pytest.raises(B.CfdError) as e:
        B.Context([(4, 8, 8)], [], case.params)
    assert e.value.code == -1
    missing = [dict(f) for f in case.faces][:-1]  # one face without a descriptor
    with pytest.raises(B.CfdError) as e:
        B.Context(case.dims, missing, case.params)
    assert e.value.code == -2
    oneway = [dict(f) for f in case.faces]
    oneway[0]["nbr_face"], oneway[0]["type"] = oneway[0]["nbr_face"], W.INTERFACE
    oneway[1]["nbr_block"] = 0
    oneway[1]["nbr_face"] = oneway[1]["face"]  # points at itself instead of back at face 0
    with pytest.raises(B.CfdError) as e:
        B.Context(case.dims, oneway, case.params)
    assert e.value.code == -2
    thin = W.c5_cylinder(ni=16, nj=6, nk=8, ratio=1.3, r_out=4.0)  # 6 nodes normal to the wall: the mirror would read a ghost
    with pytest.raises(B.CfdError) as e:
        B.Context(thin.dims, thin.faces, thin.params)
    assert e.value.code == -2
    # left-handed grid -> J < 0
    flipped = W.c1_vortex(8)
    flipped.xyz[0] = flipped.xyz[0][:, :, :, ::-1].copy()
    for f in flipped.faces:
        if f["face"] in (0, 1):
            f["shift"] = [-f["shift"][0], 0.0, 0.0]
    g2 = B.Context(flipped.dims, flipped.faces, flipped.params)
    with pytest.raises(B.CfdError) as e:
        g2.load_case(flipped)
    assert e.value.code == -3


# ------------------------------------------------------------------------------------------------
# e2e entry with host buffers (bench.py's e2e leg) and the per-kernel event timing
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("which", ["ragged-ns", "multiblock", "cylinder"])
def test_step_host_matches_oracle_and_device_path(po, W, B, which):
    import torch

    if which == "ragged-ns":
        case = ragged_case(W, 1)
    elif which == "multiblock":
        case = W.c4_multiblock(nb=10, mach=0.3)
    else:
        case = W.c5_cylinder(ni=40, nj=24, nk=10)
    o, g = pair(po, B, case)
    dt = o.cfl_dt(0.5)
    qh = [torch.from_numpy(np.ascontiguousarray(case.q0[b])).pin_memory() for b in range(len(case.dims))]
    qo = [torch.empty_like(q).pin_memory() for q in qh]
    rg = g.step_host(qh, qo, dt, want_res=True)
    ro = o.step(dt)
    assert np.allclose(rg, ro, rtol=1e-10)
    for b in range(len(case.dims)):
        ref = o.interior(b, "q")
        err = np.abs(qo[b].numpy() - ref).max() / np.abs(ref).max()
        assert err < 1e-12, (which, b, err)
        assert np.array_equal(qo[b].numpy(), g.to_numpy(b, "q"))  # D2H copy is the device state, bit for bit
    # wrong shape / non-contiguous host buffers are refused before any copy
    with pytest.raises(B.CfdError):
        g.step_host([q[:, 1:] for q in qh], qo, dt)


def test_profile_counts_every_hot_path_launch(po, W, B):
    case = ragged_case(W, 1)
    g = B.Context(case.dims, case.faces, case.params)
    g.load_case(case)
    g.profile_enable(True)
    l0 = g.launch_count
    g.step(1e-3)
    prof = g.profile_read()
    assert sum(n for _, n in prof.values()) == g.launch_count - l0
    assert all(ms >= 0.0 for ms, _ in prof.values())
    assert any(k.startswith("inviscid") or k.startswith("rhs") or k.startswith("sweep") for k in prof)
    g.profile_enable(False)
    g.step(1e-3)
    assert g.profile_read() == {}


# ------------------------------------------------------------------------------------------------
# NEXT-2: on-device CFL time step (cfd_cfl_dt) against the oracle's cfl_dt (pinned by hand formula in
# tests/test_oracle_bc_pins.py); MAX is order-independent, so the tolerance only covers sqrt / division rounding.
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("which", ["c1", "multiblock", "cylinder", "ragged"])
def test_cfl_dt_matches_oracle(po, W, B, which):
    import torch

    case = {"c1": lambda: W.c1_vortex(32), "multiblock": lambda: W.c4_multiblock(nb=12, mach=0.3),
            "cylinder": lambda: W.c5_cylinder(ni=64, nj=24, nk=10, ratio=1.15, r_out=10.0, noise=1e-2),
            "ragged": lambda: ragged_case(W, 1)}[which]()
    o, g = pair(po, B, case)
    for cfl in (0.5, 1.0):
        assert abs(g.cfl_dt(cfl) / o.cfl_dt(cfl) - 1) < 1e-13
    # after two steps (state no longer the analytic field; buffer roles exchanged by the fused stages)
    dt = o.cfl_dt(0.5)
    for _ in range(2):
        o.step(dt)
        g.step(dt)
    assert abs(g.cfl_dt(0.5) / o.cfl_dt(0.5) - 1) < 1e-13
    # local time step: cfl / s_i at interior points, its minimum is the global dt; ghosts untouched
    loc = [torch.full((nk + 2 * NG, nj + 2 * NG, ni + 2 * NG), -1.0, dtype=torch.float64, device="cuda") for (ni, nj, nk) in case.dims]
    dtg = g.cfl_dt(0.5, dt_local=loc)
    mins = []
    for b, a in enumerate(loc):
        inner = a[NG:-NG, NG:-NG, NG:-NG]
        assert (inner > 0).all()
        mins.append(float(inner.min()))
        a[NG:-NG, NG:-NG, NG:-NG] = -1.0
        assert (a == -1.0).all()
    assert abs(min(mins) / dtg - 1) < 1e-15
    with pytest.raises(B.CfdError):
        g.cfl_dt(0.0)


@pytest.mark.parametrize("bad", ["negative-pressure", "negative-density-and-pressure", "nan"])
def test_cfl_dt_refuses_a_single_non_physical_point(W, B, bad):
    """One bad interior point among 32^3 good ones must surface as CFD_E_ARG (include/cfd.h), not be dropped by the MAX
    reduction: c = sqrt(gamma p / rho) is NaN for p < 0, and real again when rho and p are both negative."""
    case = W.c1_vortex(32)
    g = B.Context(case.dims, case.faces, case.params)
    g.load_case(case)
    good = g.cfl_dt(0.5)
    assert good > 0
    q = g.interior(0, "q")
    k, j, i = 17, 5, 29  # not in the first thread / first CTA of the reduction
    if bad == "negative-pressure":
        q[4, k, j, i] = 0.25 * (q[1, k, j, i] ** 2) / q[0, k, j, i]  # e below the kinetic energy: p < 0
    elif bad == "negative-density-and-pressure":
        q[0, k, j, i] = -q[0, k, j, i]
        q[4, k, j, i] = -q[4, k, j, i]
    else:
        q[2, k, j, i] = float("nan")
    with pytest.raises(B.CfdError) as e:
        g.cfl_dt(0.5)
    assert e.value.code == -1 and "not physical" in str(e.value)
    # the context stays usable once the state is repaired
    g.interior(0, "q").copy_(__import__("torch").from_numpy(np.ascontiguousarray(case.q0[0])))
    assert g.cfl_dt(0.5) == good


# ------------------------------------------------------------------------------------------------
# NEXT-3: Sutherland viscosity mu(T) and a shocked workload (shock-vortex slab on the seeded wavy periodic grid)
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("which", ["tgv-sutherland", "ragged-sutherland", "cylinder-sutherland"])
def test_rhs_parity_sutherland(po, W, B, which):
    case = {"tgv-sutherland": lambda: W.tgv_sine_box(24, viscous=1, mach=0.4),
            "ragged-sutherland": lambda: ragged_case(W, 1),
            "cylinder-sutherland": lambda: W.c5_cylinder(ni=64, nj=24, nk=10, ratio=1.15, r_out=10.0, noise=1e-2)}[which]()
    case.params["sutherland"] = 110.4 / 288.15
    case.params["reynolds"] = 50.0   # viscous terms large enough that mu(T) matters at the 1e-12 level
    o, g = pair(po, B, case)
    assert_rhs_parity(o, g, case)
    if not which.startswith("ragged"):
        return  # T = 1 in the TGV field, ~1 around the cylinder: mu(T) ~ 1 there; the ragged field has T varying by 25 %
    # not vacuous: constant mu gives a different R
    case.params["sutherland"] = 0.0
    o0 = po.Oracle(case.dims, case.faces, case.params)
    o0.load_case(case)
    o0.rhs()
    assert np.abs(o0.interior(0, "r") - o.interior(0, "r")).max() > 1e-7 * np.abs(o.interior(0, "r")).max()


@pytest.mark.parametrize("which", ["ns-sutherland", "euler", "ns-scheme1"])
def test_shock_vortex_fifty_steps(po, W, B, which):
    """Shocked workload (pressure ratio 6, density ratio 4: shock Mach ~1.35, steps that cut the wavy grid obliquely),
    50 RK3 steps at CFL 0.5: RHS parity at the start and at the end, state parity after the 50 steps.
    Tolerance 1e-10 max|Q| on the state: the per-RHS difference is ~1e-14 of the flux scale (rounding order, FMAs,
    <= 2 ulp reciprocals); through the nonlinear weights alpha = 1/(eps + beta)^2 a perturbation d of the data changes a
    weight by O(d / (eps + beta)), beta = O(1) at the jumps and eps = 1e-6 in smooth regions where the candidates differ
    by O(h^3), so per step the difference grows like in the smooth cases; 150 stages keep it below 1e-11 in practice."""
    case = W.shock_vortex(48, viscous=0 if which == "euler" else 1)
    if which == "ns-scheme1":
        case.params["scheme"] = 1
    o, g = pair(po, B, case)
    assert_rhs_parity(o, g, case)
    dt = o.cfl_dt(0.5)
    assert abs(g.cfl_dt(0.5) / dt - 1) < 1e-13
    for _ in range(50):
        ro = o.step(dt)
        rg = g.step(dt, want_res=True)
    qo, qg = o.interior(0, "q"), g.to_numpy(0, "q")
    assert np.isfinite(qg).all()
    assert np.abs(qg - qo).max() < 1e-10 * np.abs(qo).max()
    assert np.allclose(rg, ro, rtol=1e-8)
    # the shock is still there: density jumps by > 30 % between neighbouring nodes somewhere
    rho = qo[0]
    assert (np.abs(np.diff(rho, axis=2)) / rho[:, :, 1:]).max() > 0.15
    assert_rhs_parity(o, g, case)


# ---------------------------------------------------------------------------------------------------------------------
# cfd_profile_only: the measurement aid of profiles/r2_power.md (one kernel class looped alone)
# ---------------------------------------------------------------------------------------------------------------------
def test_profile_only_masks_kernel_classes_and_default_restores_parity(po, W, B):
    case = W.c3_tgv(24)
    o, g = pair(po, B, case)
    g.field(0, "r").fill_(-7.0)
    n0 = g.launch_count
    g.profile_only(0)               # nothing of the hot classes runs: r stays untouched
    g.rhs()
    assert g.launch_count == n0
    assert float(g.interior(0, "r").min()) == -7.0 and float(g.interior(0, "r").max()) == -7.0
    assert "INVALID" in B.lib.cfd_last_error(g.h).decode()   # rc 0, but the context says the result is not one
    g.profile_only(1 << 0)          # the xi sweep alone: one launch, r = X^xi only (not the RHS)
    g.rhs()
    assert g.launch_count == n0 + 1
    assert float(g.interior(0, "r").abs().max()) != 7.0
    assert "INVALID" in B.lib.cfd_last_error(g.h).decode()
    g.profile_only()                # default: all classes, and the RHS meets the oracle again
    assert B.lib.cfd_last_error(g.h).decode() == ""
    assert_rhs_parity(o, g, case)


@pytest.mark.parametrize("tile", [0, 1, 2])
def test_visc_tile_geometries_agree_bit_for_bit_and_meet_the_oracle(po, W, B, tile):
    """cfd_set_visc_tile: the three tile geometries of k_visc_march (64 x 8, 70 x 7, 54 x 9 threads) on a ragged block that
    spans several tiles of each: the cylinder recipe (wall + far field) at 150 x 21 x 17."""
    case = W.c5_cylinder(ni=150, nj=21, nk=17)
    o, g = pair(po, B, case)
    g.set_visc_tile(tile)
    assert_rhs_parity(o, g, case)
    r_t = g.to_numpy(0, "r").copy()
    g.set_visc_tile(0)
    g.rhs()
    assert np.array_equal(g.to_numpy(0, "r"), r_t)
    g.set_visc_tile(-1)


# ---------------------------------------------------------------------------------------------------------------------
# Physical BCs next to block interfaces: the cylinder cut along the azimuth (INTERFACE faces beside WALL / FARFIELD)
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("nblk", [2, 3])
def test_split_cylinder_parity_and_equality_with_single_block(po, W, B, nblk):
    multi = W.c5_cylinder_split(nblk, ni=96, nj=20, nk=10, noise=1e-2)
    single = multi.meta["single"]
    om, gm = pair(po, B, multi)
    assert_rhs_parity(om, gm, multi)
    g1 = B.Context(single.dims, single.faces, single.params)
    g1.load_case(single)
    dt = om.cfl_dt(0.5)
    for _ in range(4):
        ro = om.step(dt)
        rg = gm.step(dt, want_res=True)
        r1 = g1.step(dt, want_res=True)
    # U17a ("inner grid points"): the residual leaves out the node planes the wall / far field own, so the cut
    # cylinder reports the single block's residual (it agreed to 1e-6 only while those planes were summed)
    assert np.allclose(rg, r1, rtol=1e-12, atol=0.0)
    cat = lambda name: np.concatenate([gm.to_numpy(b, name) for b in range(nblk)], axis=-1)
    qo = np.concatenate([om.interior(b, "q") for b in range(nblk)], axis=-1)
    assert np.abs(cat("q") - qo).max() < 1e-11 * np.abs(qo).max()
    assert np.allclose(rg, ro, rtol=1e-10)
    # the multi-block GPU run equals the single-block GPU run bit for bit (S5 + S6 next to each other)
    assert np.array_equal(cat("q"), g1.to_numpy(0, "q"))
    g1.rhs()
    gm.rhs()
    assert np.array_equal(cat("r")[:, :, 1:-1], g1.to_numpy(0, "r")[:, :, 1:-1])   # BC-owned node planes excluded (see the oracle test)
    g1.close()
