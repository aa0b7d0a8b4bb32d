"""Seeded synthetic inputs (grids, initial fields, face descriptors) for the oracle AND the CUDA path.

This module holds NONE of the method's arithmetic (no metrics, fluxes, WENO, RK): it only
produces node coordinates, initial conservative fields and block-connectivity descriptors, with
the shapes / structure of the five BASELINE.json configs (SURVEY.md §8(d), C1–C5; the paper's own
workloads, P:L599 single blocks of 1–25 M points and the jet of P:L649, are not available, so
these stand in for them — see DESIGN.md "Input recipe").  Both `oracle/` and the CUDA binding are
fed from here; neither imports the other.

Array layout everywhere: SoA [var][k][j][i] (i fastest) WITHOUT ghosts in this module; the
consumers embed the interior into their ghosted arrays (NG = 6 on every face).
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass, field

import numpy as np

GAMMA = 1.4
SEED0 = 20060796_0  # config k uses SEED0 + k

PERIODIC, INTERFACE, WALL, FARFIELD = 1, 2, 3, 4


@dataclass
class Case:
    name: str
    dims: list            # [(ni, nj, nk)] per block
    xyz: list             # [ndarray (3, nk, nj, ni)] per block
    q0: list              # [ndarray (5, nk, nj, ni)] per block
    faces: list           # [dict(block, face, type, nbr_block, nbr_face, perm, sign, shift)]
    params: dict          # gamma, mach, reynolds, prandtl, weno_eps, viscous, scheme, q_inf
    dt: float             # fixed time step for throughput runs (harness quantity, reading U16)
    steps: int
    meta: dict = field(default_factory=dict)

    @property
    def npoints(self):
        return int(sum(a * b * c for a, b, c in self.dims))


def default_params(viscous=0, mach=0.5, reynolds=1600.0, prandtl=0.71, q_inf=None, scheme=0, sutherland=0.0):
    if q_inf is None:
        q_inf = prim_to_cons(1.0, mach, 0.0, 0.0, 1.0 / GAMMA)
    return dict(gamma=GAMMA, mach=float(mach), reynolds=float(reynolds), prandtl=float(prandtl),
                weno_eps=1e-6, viscous=int(viscous), scheme=int(scheme), q_inf=[float(x) for x in q_inf],
                sutherland=float(sutherland))


def prim_to_cons(rho, u, v, w, p):
    rho, u, v, w, p = np.broadcast_arrays(*(np.asarray(a, dtype=np.float64) for a in (rho, u, v, w, p)))
    return np.stack([rho, rho * u, rho * v, rho * w, p / (GAMMA - 1.0) + 0.5 * rho * (u * u + v * v + w * w)])


def periodic_faces(block=0, L=(0.0, 0.0, 0.0)):
    """Six PERIODIC faces connecting a block to itself; L = coordinate period per axis (x,y,z shift
    carried by the xi, eta, zeta faces respectively)."""
    fs = []
    for a in range(3):
        for s in range(2):
            sh = [0.0, 0.0, 0.0]
            sh[a] = -L[a] if s == 0 else L[a]
            fs.append(dict(block=block, face=2 * a + s, type=PERIODIC, nbr_block=block, nbr_face=2 * a + (1 - s),
                           perm=[0, 1, 2], sign=[1, 1, 1], shift=sh))
    return fs


def _uniform_nodes(n, L):
    """node coordinates xi_a = i * L_a / n_a, arrays shaped (nk, nj, ni)."""
    ni, nj, nk = n
    x = np.arange(ni) * (L[0] / ni)
    y = np.arange(nj) * (L[1] / nj)
    z = np.arange(nk) * (L[2] / nk)
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    return X, Y, Z


# ------------------------------------------------------------------------------------------
# mappings
# ------------------------------------------------------------------------------------------
def c1_mapping(X, Y, Z):
    """x = xi + 0.1 sin(pi eta/5) sin(pi zeta/5), cyclic (BASELINE.json config 1)."""
    s = lambda a: np.sin(np.pi * a / 5.0)
    return np.stack([X + 0.1 * s(Y) * s(Z), Y + 0.1 * s(Z) * s(X), Z + 0.1 * s(X) * s(Y)])


def wavy_modes(seed):
    """Seeded random-phase sinusoidal warp: per coordinate 2–4 modes (a_m, b_m in 1..4, phases U[0,2pi))."""
    rng = np.random.default_rng(seed)
    modes = []
    for c in range(3):
        nc = int(rng.integers(2, 5))
        modes.append(dict(a=rng.integers(1, 5, nc), b=rng.integers(1, 5, nc),
                          phi=rng.uniform(0, 2 * np.pi, nc), psi=rng.uniform(0, 2 * np.pi, nc)))
    return modes


def wavy_mapping(X, Y, Z, L, h, modes, amp=0.2):
    """x_c = x0_c + (amp*h/n_c) sum_m sin(2 pi a_m x0_{c+1}/L + phi_m) sin(2 pi b_m x0_{c+2}/L + psi_m)."""
    x0 = [X, Y, Z]
    out = []
    for c in range(3):
        md = modes[c]
        nc = len(md["a"])
        d = np.zeros_like(X)
        for m in range(nc):
            d += np.sin(2 * np.pi * md["a"][m] * x0[(c + 1) % 3] / L + md["phi"][m]) * \
                 np.sin(2 * np.pi * md["b"][m] * x0[(c + 2) % 3] / L + md["psi"][m])
        out.append(x0[c] + (amp * h / nc) * d)
    return np.stack(out)


# ------------------------------------------------------------------------------------------
# initial fields
# ------------------------------------------------------------------------------------------
def vortex_field(xyz, t=0.0, L=10.0, strength=5.0, mach=0.5, centre=(5.0, 5.0)):
    """Isentropic vortex (axis || z) advected with (mach,0,0), a_inf = 1 units; nearest periodic image."""
    g = GAMMA
    xb = (xyz[0] - centre[0] - mach * t + 0.5 * L) % L - 0.5 * L
    yb = (xyz[1] - centre[1] + 0.5 * L) % L - 0.5 * L
    r2 = xb * xb + yb * yb
    f = strength / (2 * np.pi) * np.exp(0.5 * (1.0 - r2))
    u = mach - f * yb
    v = f * xb
    T = 1.0 - (g - 1.0) * strength ** 2 / (8 * np.pi ** 2) * np.exp(1.0 - r2)
    rho = T ** (1.0 / (g - 1.0))
    p = rho * T / g
    return prim_to_cons(rho, u, v, 0.0 * u, p)


def density_wave_field(xyz, t=0.0, L=10.0, vel=(0.5, 0.3, 0.2), amp=0.2):
    """rho = 1 + amp sin(2 pi (x+y+z - (u+v+w) t)/L), constant velocity and pressure: exact Euler solution."""
    s = xyz[0] + xyz[1] + xyz[2] - (vel[0] + vel[1] + vel[2]) * t
    rho = 1.0 + amp * np.sin(2 * np.pi * s / L)
    one = np.ones_like(rho)
    return prim_to_cons(rho, vel[0] * one, vel[1] * one, vel[2] * one, one / GAMMA)


def tgv_field(xyz, mach=0.1):
    """Taylor–Green vortex, T = 1 (rho = gamma p), a_inf = 1 units."""
    x, y, z = xyz
    u = mach * np.sin(x) * np.cos(y) * np.cos(z)
    v = -mach * np.cos(x) * np.sin(y) * np.cos(z)
    p = 1.0 / GAMMA + mach ** 2 / 16.0 * (np.cos(2 * x) + np.cos(2 * y)) * (np.cos(2 * z) + 2.0)
    rho = GAMMA * p
    return prim_to_cons(rho, u, v, 0.0 * u, p)


# ------------------------------------------------------------------------------------------
# the five configs (+ helpers); every size is a parameter so tests can run reduced copies
# ------------------------------------------------------------------------------------------
def c1_vortex(n=32, steps=10):
    L = 10.0
    X, Y, Z = _uniform_nodes((n, n, n), (L, L, L))
    xyz = c1_mapping(X, Y, Z)
    q0 = vortex_field(xyz)
    h = L / n
    return Case("C1-vortex", [(n, n, n)], [xyz], [q0], periodic_faces(0, (L, L, L)),
                default_params(viscous=0, mach=0.5), dt=0.5 * h / 2.6, steps=steps, meta=dict(L=L, h=h))


def density_wave(n=16, mapping="c1"):
    L = 10.0
    X, Y, Z = _uniform_nodes((n, n, n), (L, L, L))
    xyz = c1_mapping(X, Y, Z) if mapping == "c1" else np.stack([X, Y, Z])
    q0 = density_wave_field(xyz)
    h = L / n
    return Case("density-wave", [(n, n, n)], [xyz], [q0], periodic_faces(0, (L, L, L)),
                default_params(viscous=0, mach=0.5), dt=0.2 * h ** (5.0 / 3.0), steps=0, meta=dict(L=L, h=h))


def wavy_box(n, seed, L=2 * np.pi, amp=0.2):
    n3 = (n, n, n) if np.isscalar(n) else tuple(n)
    X, Y, Z = _uniform_nodes(n3, (L, L, L))
    h = L / max(n3)
    modes = wavy_modes(seed)
    return wavy_mapping(X, Y, Z, L, h, modes, amp), h, modes


def c2_freestream(n=64, viscous=1, steps=100, seed=SEED0 + 2, amp=0.2):
    L = 2 * np.pi
    xyz, h, _ = wavy_box(n, seed, L, amp)
    rng = np.random.default_rng(seed + 1000)
    d = rng.normal(size=3)
    d /= np.linalg.norm(d)
    one = np.ones(xyz.shape[1:])
    q0 = prim_to_cons(one, 0.5 * d[0] * one, 0.5 * d[1] * one, 0.5 * d[2] * one, one / GAMMA)
    qinf = prim_to_cons(1.0, 0.5 * d[0], 0.5 * d[1], 0.5 * d[2], 1.0 / GAMMA)
    return Case("C2-freestream", [tuple([n] * 3)], [xyz], [q0], periodic_faces(0, (L, L, L)),
                default_params(viscous=viscous, mach=0.5, reynolds=1600.0, q_inf=qinf),
                dt=0.5 * 0.75 * h / 1.5 / 1.8, steps=steps, meta=dict(L=L, h=h, dir=d))


def c3_tgv(n=128, viscous=1, steps=200, seed=SEED0 + 3, mach=0.1):
    L = 2 * np.pi
    xyz, h, _ = wavy_box(n, seed, L)
    q0 = tgv_field(xyz, mach)
    return Case("C3-tgv", [tuple([n] * 3)], [xyz], [q0], periodic_faces(0, (L, L, L)),
                default_params(viscous=viscous, mach=mach, reynolds=1600.0, prandtl=0.71),
                dt=0.5 * 0.75 * h / (1.0 + mach) / 1.8, steps=steps, meta=dict(L=L, h=h))


# ---- proper signed permutations (24 rotations of the cube) ----------------------------------
def proper_rotations():
    out = []
    for perm in itertools.permutations(range(3)):
        par = 1 if perm in ((0, 1, 2), (1, 2, 0), (2, 0, 1)) else -1
        for sg in itertools.product((1, -1), repeat=3):
            if par * sg[0] * sg[1] * sg[2] == 1:
                out.append((perm, sg))
    return out


def _global_index(origin, nb, gax, gsg, G):
    """Global (K, J, I) index arrays, shaped (n2, n1, n0), of a block whose local axis a runs along global
    axis gax[a] in direction gsg[a] starting at `origin` (periodic wrap)."""
    l2, l1, l0 = np.meshgrid(np.arange(nb[2]), np.arange(nb[1]), np.arange(nb[0]), indexing="ij")
    loc = [l0, l1, l2]
    gidx = [None, None, None]
    for a in range(3):
        A = gax[a]
        r = loc[a] if gsg[a] > 0 else nb[a] - 1 - loc[a]
        gidx[A] = (origin[A] + r) % G[A]
    return gidx[2], gidx[1], gidx[0]


def _extract_block(Garr, origin, nb, gax, gsg):
    """Cut a block out of a global periodic array Garr[..., K, J, I] -> [..., l2, l1, l0]."""
    G = Garr.shape[-3:][::-1]
    gk, gj, gi = _global_index(origin, nb, gax, gsg, G)
    return np.ascontiguousarray(Garr[..., gk, gj, gi])


def split_periodic(xyz_g, q_g, L, nblk=(2, 2, 2), rotations=None):
    """Tile a global periodic single-block grid into nblk blocks whose local axes are signed permutations
    of the global ones; returns dims, xyz, q0, faces and the bookkeeping needed to map back."""
    G = xyz_g.shape[1:][::-1]  # (GI, GJ, GK)
    nbs = [G[a] // nblk[a] for a in range(3)]
    assert all(nbs[a] * nblk[a] == G[a] for a in range(3))
    blocks = list(itertools.product(range(nblk[0]), range(nblk[1]), range(nblk[2])))
    nblocks = len(blocks)
    if rotations is None:
        rotations = [((0, 1, 2), (1, 1, 1))] * nblocks
    bid = {bc: n for n, bc in enumerate(blocks)}
    dims, xyz, q0, info = [], [], [], []
    for n, bc in enumerate(blocks):
        gax, gsg = list(rotations[n][0]), list(rotations[n][1])
        origin = [bc[A] * nbs[A] for A in range(3)]
        nb_local = [nbs[gax[a]] for a in range(3)]
        dims.append(tuple(nb_local))
        xyz.append(_extract_block(xyz_g, origin, nb_local, gax, gsg))
        q0.append(_extract_block(q_g, origin, nb_local, gax, gsg))
        info.append(dict(origin=origin, gax=gax, gsg=gsg, n=nb_local))
    faces = []
    for n, bc in enumerate(blocks):
        gax, gsg = info[n]["gax"], info[n]["gsg"]
        for a in range(3):
            for s in range(2):
                A = gax[a]
                S = s if gsg[a] > 0 else 1 - s
                nbc = list(bc)
                nbc[A] = (bc[A] + (1 if S == 1 else -1)) % nblk[A]
                wrap = (S == 1 and bc[A] == nblk[A] - 1) or (S == 0 and bc[A] == 0)
                m = bid[tuple(nbc)]
                gax2, gsg2 = info[m]["gax"], info[m]["gsg"]
                perm = [gax2.index(gax[b]) for b in range(3)]
                sign = [gsg[b] * gsg2[perm[b]] for b in range(3)]
                ap = perm[a]
                sp = (1 - S) if gsg2[ap] > 0 else S
                shift = [0.0, 0.0, 0.0]
                if wrap:
                    shift[A] = L[A] if S == 1 else -L[A]
                faces.append(dict(block=n, face=2 * a + s, type=PERIODIC if wrap else INTERFACE, nbr_block=m,
                                  nbr_face=2 * ap + sp, perm=perm, sign=sign, shift=shift))
    return dims, xyz, q0, faces, info


def gather_blocks(arrs, info, G):
    """Inverse of split_periodic for interior arrays [nv, l2, l1, l0] -> global [nv, GK, GJ, GI]."""
    nv = arrs[0].shape[0]
    out = np.zeros((nv, G[2], G[1], G[0]))
    for a, inf in zip(arrs, info):
        gk, gj, gi = _global_index(inf["origin"], inf["n"], inf["gax"], inf["gsg"], G)
        out[:, gk, gj, gi] = a
    return out


def c4_multiblock(nb=96, viscous=1, steps=100, seed=SEED0 + 4, mach=0.1, permute=True, wavy=True):
    """8 point-matched blocks of nb^3 tiling a periodic (2 nb)^3 node grid on [0,2pi]^3, each with a seeded
    proper signed permutation of the global axes; TGV field; 24 interfaces incl. periodic wraps."""
    L = 2 * np.pi
    G = 2 * nb
    if wavy:
        xyz_g, h, _ = wavy_box(G, seed, L)
    else:
        X, Y, Z = _uniform_nodes((G, G, G), (L, L, L))
        xyz_g, h = np.stack([X, Y, Z]), L / G
    q_g = tgv_field(xyz_g, mach)
    rng = np.random.default_rng(seed + 1000)
    rots = proper_rotations()
    rotations = [rots[int(rng.integers(0, 24))] for _ in range(8)] if permute else None
    dims, xyz, q0, faces, info = split_periodic(xyz_g, q_g, (L, L, L), (2, 2, 2), rotations)
    return Case("C4-multiblock", dims, xyz, q0, faces,
                default_params(viscous=viscous, mach=mach, reynolds=1600.0, prandtl=0.71),
                dt=0.5 * 0.75 * h / (1.0 + mach) / 1.8, steps=steps,
                meta=dict(L=L, h=h, info=info, G=(G, G, G), xyz_g=xyz_g, q_g=q_g))


def c5_cylinder(ni=1024, nj=256, nk=128, ratio=1.02, r_out=20.0, steps=50, seed=SEED0 + 5, mach=0.2,
                reynolds=3900.0, noise=1e-4, viscous=1):
    """Cylinder O-grid: xi = azimuth (periodic, clockwise so that J > 0), eta = radius (geometric stretching,
    WALL at j=0, FARFIELD at j=nj-1), zeta = span (periodic, Lz = pi)."""
    Lz = np.pi
    dr0 = (r_out - 0.5) * (ratio - 1.0) / (ratio ** (nj - 1) - 1.0)
    r = 0.5 + dr0 * (ratio ** np.arange(nj) - 1.0) / (ratio - 1.0)
    th = -2 * np.pi * np.arange(ni) / ni
    z = np.arange(nk) * (Lz / nk)
    Zz, R, TH = np.meshgrid(z, r, th, indexing="ij")
    xyz = np.stack([R * np.cos(TH), R * np.sin(TH), Zz])
    rng = np.random.default_rng(seed)
    one = np.ones(xyz.shape[1:])
    nz = lambda: rng.uniform(-noise, noise, size=one.shape)
    q0 = prim_to_cons(one, mach + nz(), nz(), nz(), one / GAMMA)
    qinf = prim_to_cons(1.0, mach, 0.0, 0.0, 1.0 / GAMMA)
    faces = []
    for s in range(2):
        faces.append(dict(block=0, face=s, type=PERIODIC, nbr_block=0, nbr_face=1 - s, perm=[0, 1, 2], sign=[1, 1, 1],
                          shift=[0.0, 0.0, 0.0]))
    faces.append(dict(block=0, face=2, type=WALL, nbr_block=-1, nbr_face=-1, perm=[0, 1, 2], sign=[1, 1, 1], shift=[0.0] * 3))
    faces.append(dict(block=0, face=3, type=FARFIELD, nbr_block=-1, nbr_face=-1, perm=[0, 1, 2], sign=[1, 1, 1], shift=[0.0] * 3))
    for s in range(2):
        faces.append(dict(block=0, face=4 + s, type=PERIODIC, nbr_block=0, nbr_face=5 - s, perm=[0, 1, 2], sign=[1, 1, 1],
                          shift=[0.0, 0.0, -Lz if s == 0 else Lz]))
    hmin = min(dr0, 0.5 * 2 * np.pi / ni, Lz / nk)
    return Case("C5-cylinder", [(ni, nj, nk)], [xyz], [q0], faces,
                default_params(viscous=viscous, mach=mach, reynolds=reynolds, prandtl=0.71, q_inf=qinf),
                dt=0.5 * hmin / (1.0 + mach) / 1.8, steps=steps, meta=dict(dr0=dr0, hmin=hmin))


def c5_cylinder_split(nblk=2, **kw):
    """The cylinder of c5_cylinder cut along the azimuth into nblk point-matched blocks (INTERFACE faces in xi, also across
    theta = 0; WALL / FARFIELD in eta and the periodic span in zeta on every block): physical boundary conditions next to
    block interfaces, the case the paper's bc_block + bc_phys order is for (Fig. 2).  Same nodes and field as
    the single block, so the two runs must agree point for point."""
    one = c5_cylinder(**kw)
    ni, nj, nk = one.dims[0]
    if ni % nblk or ni // nblk < 6:
        raise ValueError("c5_cylinder_split: ni must be a multiple of nblk with at least 6 nodes per block")
    nb = ni // nblk
    Lz = np.pi
    dims, xyz, q0, faces = [], [], [], []
    for b in range(nblk):
        sl = slice(b * nb, (b + 1) * nb)
        dims.append((nb, nj, nk))
        xyz.append(np.ascontiguousarray(one.xyz[0][..., sl]))
        q0.append(np.ascontiguousarray(one.q0[0][..., sl]))
        eye = dict(perm=[0, 1, 2], sign=[1, 1, 1])
        faces.append(dict(block=b, face=0, type=INTERFACE, nbr_block=(b - 1) % nblk, nbr_face=1, shift=[0.0] * 3, **eye))
        faces.append(dict(block=b, face=1, type=INTERFACE, nbr_block=(b + 1) % nblk, nbr_face=0, shift=[0.0] * 3, **eye))
        faces.append(dict(block=b, face=2, type=WALL, nbr_block=-1, nbr_face=-1, shift=[0.0] * 3, **eye))
        faces.append(dict(block=b, face=3, type=FARFIELD, nbr_block=-1, nbr_face=-1, shift=[0.0] * 3, **eye))
        for s2 in range(2):
            faces.append(dict(block=b, face=4 + s2, type=PERIODIC, nbr_block=b, nbr_face=5 - s2,
                              shift=[0.0, 0.0, -Lz if s2 == 0 else Lz], **eye))
    return Case(f"C5-cylinder-{nblk}-blocks", dims, xyz, q0, faces, dict(one.params), dt=one.dt, steps=one.steps,
                meta=dict(one.meta, nblk=nblk, single=one))


def sweep_block(n=256, viscous=1, seed=SEED0 + 3, mach=0.1):
    """Throughput sweep block (256^3 / 384^3 / 512^3): C3's mapping and field (SURVEY §8(d) 'Sweep')."""
    c = c3_tgv(n=n, viscous=viscous, steps=20, seed=seed, mach=mach)
    c.name = f"sweep-{n}^3-{'ns' if viscous else 'euler'}"
    return c


def tgv_sine_box(n=16, viscous=1, mach=0.1, amp=0.1):
    """TGV on [0,2pi]^3 with the analytic warp x = xi + amp sin(eta) sin(zeta) (cyclic) — the grid of
    SURVEY.md Appendix A.2 (survey-time cross-check values)."""
    L = 2 * np.pi
    X, Y, Z = _uniform_nodes((n, n, n), (L, L, L))
    xyz = np.stack([X + amp * np.sin(Y) * np.sin(Z), Y + amp * np.sin(Z) * np.sin(X), Z + amp * np.sin(X) * np.sin(Y)])
    q0 = tgv_field(xyz, mach)
    h = L / n
    return Case("tgv-sine-box", [(n, n, n)], [xyz], [q0], periodic_faces(0, (L, L, L)),
                default_params(viscous=viscous, mach=mach, reynolds=1600.0, prandtl=0.71),
                dt=0.5 * 0.75 * h / (1.0 + mach) / 1.8, steps=0, meta=dict(L=L, h=h))


def shock_vortex(n=48, viscous=1, sutherland=110.4 / 288.15, seed=SEED0 + 6, pressure_ratio=6.0, density_ratio=4.0,
                 strength=1.5, reynolds=500.0, steps=50):
    """Shocked periodic workload (the paper's target flows are supersonic jets): a
    high-pressure slab x in [L/4, 3L/4) of the seeded wavy periodic box (two shock / contact / rarefaction systems, the
    initial jumps are steps that cut the curvilinear grid lines obliquely) with an isentropic vortex (axis || z, radius
    scale 0.5) inside the slab and a weak spanwise velocity, so that the nonlinear WENO weights work far from the smooth
    limit in all three sweeps (shock Mach number ~ 1.35 for the default jumps; ratios of 10 / 8 blow up with this
    scheme's unlimited central terms).  Navier–Stokes with Sutherland viscosity (or Euler with viscous=0)."""
    L = 2 * np.pi
    xyz, h, _ = wavy_box(n, seed, L)
    x, y, z = xyz
    g = GAMMA
    inside = (x % L >= 0.25 * L) & (x % L < 0.75 * L)
    rho_b = np.where(inside, 1.0, 1.0 / density_ratio)
    p_b = np.where(inside, 1.0 / g, 1.0 / (g * pressure_ratio))
    T_b = g * p_b / rho_b
    r0 = 0.5
    xb = (x - 0.5 * L) / r0
    yb = ((y - 0.5 * L + 0.5 * L) % L - 0.5 * L) / r0
    r2 = xb * xb + yb * yb
    f = strength / (2 * np.pi) * np.exp(0.5 * (1.0 - r2))
    u = -f * yb
    v = f * xb
    w = 0.05 * np.sin(z) * np.cos(y)
    T = T_b * (1.0 - (g - 1.0) * strength ** 2 / (8 * np.pi ** 2) * np.exp(1.0 - r2))
    rho = rho_b * (T / T_b) ** (1.0 / (g - 1.0))
    p = rho * T / g
    q0 = prim_to_cons(rho, u, v, w, p)
    prm = default_params(viscous=viscous, mach=1.0, reynolds=reynolds, prandtl=0.71, sutherland=sutherland if viscous else 0.0)
    return Case("shock-vortex", [tuple([n] * 3)], [xyz], [q0], periodic_faces(0, (L, L, L)), prm,
                dt=0.4 * 0.75 * h / 2.2 / 1.8, steps=steps, meta=dict(L=L, h=h))
