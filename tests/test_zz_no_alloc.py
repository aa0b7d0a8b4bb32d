"""cfd_rk_stage1_static -- the entry point for callers that cannot allocate device memory -- against the existing path.

Some users of the library cannot call cudaMalloc and cannot hand over a workspace: a solver plug-in inside an application
whose own arena already holds all of the GPU's memory (cudaMalloc fails there), a coupling loop that may not stall the
device (cudaMalloc / cudaFree synchronise against all streams), a callback that only receives q and r.  For them RK3
stage 1 + the residual sum exists as a context-free call whose scratch (the per-CTA partial sums) is a fixed array inside
the library, shared by all calls on a device and never cleared.  What this file checks is therefore exactly what could go
wrong with that: the values must be those of cfd_rk_stage(ctx, 1, ...) (the tests' tolerance for the residual is
rtol 1e-12; the state is compared bit for bit), and a SECOND call right after the first -- on a smaller block, so that the
array still holds the first call's partial sums beyond the range the second one uses -- must be just as right.

This file is collected last (test_zz_*): `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests proper.  It passes alone in a fresh process (the first call does the per-device set-up) and after the others.
"""
import ctypes as C

import numpy as np
import pytest

NG = 6


def _wavy_case(W, n, seed):
    """One periodic wavy block of n = (ni, nj, nk) interior points with a smooth non-uniform state."""
    L = 2 * np.pi
    X, Y, Z = W._uniform_nodes(n, (L, L, L))
    xyz = W.wavy_mapping(X, Y, Z, L, L / max(n), W.wavy_modes(seed), amp=0.2)
    q0 = W.tgv_field(xyz, 0.4)
    q0 = W.prim_to_cons(q0[0] * (1 + 0.1 * np.sin(xyz[1])), q0[1] / q0[0] + 0.2, q0[2] / q0[0], 0.1 * np.cos(xyz[0] + xyz[2]),
                        (1 / 1.4) * (1 + 0.05 * np.cos(xyz[2])))
    return W.Case("no-alloc", [n], [xyz], [q0], W.periodic_faces(0, (L, L, L)),
                  W.default_params(viscous=1, mach=0.4, reynolds=300.0), dt=1e-3, steps=0)


@pytest.mark.gpu
def test_static_scratch_stage1_matches_context_path_on_consecutive_calls(W):
    import torch

    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2006_07964_b200 import binding as B

    dt = 1.7e-3
    # 32^3 = 128 CTAs of partial sums; then 71 x 23 x 15 = 96 CTAs with a ragged last CTA (slots 96..127 keep call 1's sums);
    # then the first size again with another state
    for call, (n, seed) in enumerate([((32, 32, 32), 3), ((71, 23, 15), 11), ((32, 32, 32), 5)]):
        case = _wavy_case(W, n, seed)
        g = B.Context(case.dims, case.faces, case.params)
        g.load_case(case)
        g.rhs()
        # the new entry point works on private copies (ghost layers included) of what the existing path is about to consume
        q = g.field(0, "q").clone()
        r = g.field(0, "r").clone()
        qn = torch.full_like(q, float("nan"))
        res = torch.full((5,), float("nan"), dtype=torch.float64, device=q.device)
        q_before = q.clone()

        want_res = g.rk_stage(1, dt, want_res=True)  # existing path: context + caller-allocated workspace
        B.rk_stage1_static(q, qn, r, n, dt, res)      # new path: no context, no workspace, no allocation in the library
        torch.cuda.synchronize()

        got_res = res.cpu().numpy()
        assert np.all(np.isfinite(got_res)) and np.all(want_res > 0)
        assert np.allclose(got_res, want_res, rtol=1e-12, atol=0.0), (call, got_res, want_res)
        I = (slice(None), slice(NG, -NG), slice(NG, -NG), slice(NG, -NG))
        assert torch.equal(q[I], g.field(0, "q")[I]), call
        assert torch.equal(qn[I], g.field(0, "qn")[I]), call
        # ghost layers are not the entry point's business: q's are untouched, qn's never written
        ghost = torch.ones_like(q, dtype=torch.bool)
        ghost[I] = False
        assert torch.equal(q[ghost], q_before[ghost])
        assert bool(torch.isnan(qn[ghost]).all())
        g.close()


def test_static_scratch_entry_rejects_what_it_cannot_hold():
    """Argument checks come before any CUDA call, so they run without a GPU: a block beyond CFD_STATIC_MAX_POINTS is refused
    with CFD_E_WORKSPACE and a message naming the limit; null pointers and empty sizes give CFD_E_ARG."""
    from paper_2006_07964_b200 import binding as B

    L = B.lib
    fake = C.c_void_p(4096)  # never dereferenced: the call must fail before it touches device memory
    assert B.STATIC_MAX_POINTS == 128 ** 3
    rc = L.cfd_rk_stage1_static(fake, fake, fake, 128, 128, 129, 1e-3, fake, None)
    assert rc == -5
    msg = L.cfd_static_last_error().decode()
    assert "CFD_STATIC_MAX_POINTS" in msg and "2113536" in msg and "2097152" in msg, msg
    assert L.cfd_rk_stage1_static(None, fake, fake, 8, 8, 8, 1e-3, fake, None) == -1
    assert "null" in L.cfd_static_last_error().decode()
    assert L.cfd_rk_stage1_static(fake, fake, fake, 8, 0, 8, 1e-3, fake, None) == -1
    assert L.cfd_rk_stage1_static(C.c_void_p(4100), fake, fake, 8, 8, 8, 1e-3, fake, None) == -1
    # the header's constants and the library agree
    src = open(B.HERE + "/../include/cfd.h").read()
    assert "#define CFD_STATIC_MAX_POINTS 2097152" in src and "#define CFD_STATIC_SCRATCH_BYTES 327680" in src
