"""GPU parity of the tracer particles (Sec. VI, Eq. 20-22) against the CPU oracle, through the C ABI.

Tolerances: the cell index floor(x N/L) is an integer decided in fp64 on both sides from the same expression; the
push itself is ~150 fp64 operations, so positions and velocities agree to a few ulp per step: after n steps the
bound used is 1e-13 * (1 + n) relative to L resp. |v| (round-off grows linearly at worst; a flipped cell decision at
an exact cell boundary changes nothing because CIC is continuous across cells)."""
import math

import numpy as np
import pytest

from paper_1810_12707_b200 import inputs

pytestmark = pytest.mark.gpu
L = 2 * math.pi


@pytest.fixture(scope="module")
def MHD():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1810_12707_b200 import build, binding
    build.build()
    return binding.MHD


def particles(n, seed, vscale=1.0):
    rng = np.random.default_rng(seed)
    pos = [rng.uniform(0, L, n) for _ in range(3)]
    vel = [rng.standard_normal(n) * vscale for _ in range(3)]
    return pos, vel


def close(a, b, tol):
    return all(np.max(np.abs(x - y)) <= tol for x, y in zip(a, b))


def wrapped_diff(a, b):
    d = np.abs(a - b)
    return np.minimum(d, L - d)


@pytest.mark.parametrize("N", [16, 32, 64, 128])
def test_frozen_field_push_matches_oracle(orc, MHD, N):
    """mhd_tracers_push (one launch, nsteps pushes in the frozen B of the state) vs the oracle's loop; 5003 particles
    (ragged tail of the 128-thread blocks), velocities large enough to cross the periodic boundary many times."""
    cfg = inputs.config3(N, kmax=4) if N >= 32 else inputs.config1(N)
    g = MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, 0.05)
    g.set_fields(cfg.prim, "primitive")
    pos, vel = particles(5003, N, vscale=3.0)
    g.tracers_set(pos, vel)
    nsteps = 40
    g.tracers_push(nsteps)
    pg, vg = g.tracers_get()
    B = g.get_fields("conservative")[5:8]            # the projected state the GPU holds (identical input for both)
    po, vo = orc.tracers_push(B, pos, vel, 0.05, nsteps, L=cfg.L)
    tol = 1e-13 * (1 + nsteps)
    for c in range(3):
        assert np.max(wrapped_diff(pg[c], po[c])) <= tol * L
        assert np.max(np.abs(vg[c] - vo[c])) <= tol * 10.0
        assert np.all(pg[c] >= 0) and np.all(pg[c] < L)


def test_initial_velocity_is_cic_of_u(orc, MHD):
    cfg = inputs.config3(32, kmax=4)
    rho = 1.0 + 0.3 * np.sin(inputs.grid(32)[0])           # non-uniform density: u = m/rho at the grid points
    prim = list(cfg.prim)
    prim[0] = rho * np.ones_like(prim[0])
    g = MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt)
    g.set_fields(prim, "primitive")
    pos, _ = particles(777, 5)
    g.tracers_set(pos)
    pg, vg = g.tracers_get()
    U = g.get_fields("conservative")
    u = [U[1 + c] / U[0] for c in range(3)]
    vo = orc.cic(u, pos, L=cfg.L)
    for c in range(3):
        assert np.max(np.abs(vg[c] - vo[c])) <= 1e-13
        assert np.array_equal(pg[c], pos[c])


@pytest.mark.parametrize("N,fused", [(32, 1), (128, 1), (128, 0), (128, 2)])
def test_tracers_advance_with_the_fields(orc, MHD, N, fused):
    """mhd_step with tracers attached vs the oracle with tracers attached: the push of step n uses B(t_n).  N = 128 with
    fused = 1 takes B from the by-product of the fused x sweep, the other cases from a separate inverse transform."""
    cfg = inputs.config3(N, kmax=4) if N > 32 else inputs.config2(N)
    dt = 2e-3
    o = orc.Oracle(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, dt)
    o.set_fields(cfg.prim, "primitive")
    g = MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, dt)
    g.set_option(1, fused)
    g.set_fields(cfg.prim, "primitive")
    pos, vel = particles(1000, 11 + N, vscale=2.0)
    o.tracers_set(pos, vel)
    g.tracers_set(pos, vel)
    nsteps = 6
    o.step(nsteps)
    g.step(3)
    g.step(nsteps - 3)                                  # split calls: same result
    po, vo = o.tracers_get()
    pg, vg = g.tracers_get()
    tol = 1e-13 * (1 + nsteps)
    for c in range(3):
        assert np.max(wrapped_diff(pg[c], po[c])) <= tol * L, (c, np.max(wrapped_diff(pg[c], po[c])))
        assert np.max(np.abs(vg[c] - vo[c])) <= tol * 10.0
    # and the fields are untouched by the presence of tracers
    Ug, Uo = g.get_fields(), o.get_fields()
    scale = max(np.linalg.norm(x) for x in Uo)       # some components (m_z, B_z of config 2) are roundoff-small
    for f in range(8):
        assert np.linalg.norm(Ug[f] - Uo[f]) <= 1e-12 * scale


@pytest.mark.parametrize("integ", [1, 2])
def test_tracers_with_other_integrators_use_start_of_step_B(orc, MHD, integ):
    """RK4 / predictor-corrector: the tracers still see B(t_n) of the step's initial state (separate transform)."""
    cfg = inputs.config2(32)
    g = MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, 1e-3)
    g.set_option(3, integ)
    g.set_fields(cfg.prim, "primitive")
    pos, vel = particles(300, 2)
    g.tracers_set(pos, vel)
    p, v = pos, vel
    for s in range(3):
        B = g.get_fields("conservative")[5:8]
        p, v = orc.tracers_push(B, p, v, 1e-3, 1, L=cfg.L)
        g.step(1)
    pg, vg = g.tracers_get()
    for c in range(3):
        assert np.max(wrapped_diff(pg[c], p[c])) <= 1e-12 and np.max(np.abs(vg[c] - v[c])) <= 1e-12


def test_device_pointers_and_errors(MHD):
    import torch
    cfg = inputs.config1(32)
    g = MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt)
    pos, vel = particles(100, 3)
    with pytest.raises(RuntimeError):
        g.tracers_set(pos)                               # CIC of u needs fields
    g.set_fields(cfg.prim, "primitive")
    with pytest.raises(RuntimeError):
        g.tracers_push(1)                                # no tracers yet
    dp = [torch.from_numpy(x).cuda() for x in pos]
    dv = [torch.from_numpy(x).cuda() for x in vel]
    g.tracers_set(dp, dv)
    g.tracers_push(3)
    pd, vd = g.tracers_get("device")
    g.tracers_set(pos, vel)
    g.tracers_push(3)
    ph, vh = g.tracers_get()
    for c in range(3):
        assert np.array_equal(pd[c].cpu().numpy(), ph[c]) and np.array_equal(vd[c].cpu().numpy(), vh[c])
    # speed is conserved by the rotation
    s0 = np.sqrt(sum(x ** 2 for x in vel))
    s1 = np.sqrt(sum(x ** 2 for x in vh))
    assert np.max(np.abs(s1 - s0) / s0) <= 1e-14
    # positions outside [0, L) are wrapped on input
    far = [x + 3 * L for x in pos]
    g.tracers_set(far, vel)
    pw, _ = g.tracers_get()
    for c in range(3):
        assert np.max(wrapped_diff(pw[c], pos[c])) <= 1e-14 * 4 * L and np.all(pw[c] < L)


@pytest.mark.parametrize("flags,N,brick,slab,integ", [(0, 64, 0, 0, 0), (6, 32, 4, 5, 0), (2, 64, 7, 9, 1)])
def test_tracers_on_the_chunked_pipeline(MHD, flags, N, brick, slab, integ):
    """Tracers on an MHD_FLAG_OUT_OF_CORE context (compact storage in HBM, or state / work arrays in pinned host memory): the
    tracers keep their own real-space copy of B, filled slab by slab at the start of every step, and the initial velocity is
    the CIC interpolation of u.  Same pushes as in core: positions and velocities agree to roundoff, frozen field and
    evolving field (Adams-Bashforth and RK4)."""
    from paper_1810_12707_b200 import binding as b
    cfg = inputs.config3(N, kmax=4)
    dt = 2e-3
    extra = b.MHD_FLAG_STAGE_STORAGE if integ else 0
    ref = MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, dt)
    g = MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, dt, flags=b.MHD_FLAG_OUT_OF_CORE | flags | extra)
    g.set_option(b.MHD_OPT_OOC_BRICK, brick); g.set_option(b.MHD_OPT_OOC_SLAB, slab)
    for m in (ref, g):
        m.set_option(b.MHD_OPT_INTEGRATOR, integ)
        m.set_fields(cfg.prim, "primitive")
    pos, _ = particles(777, 5 + N)
    ref.tracers_set(pos); g.tracers_set(pos)                 # v0 = CIC of u on both
    for m in (ref, g):
        m.tracers_push(3)                                    # frozen field
        m.step(2); m.step(3)                                 # evolving field
    pr, vr = ref.tracers_get()
    pg, vg = g.tracers_get()
    for c in range(3):
        assert np.max(wrapped_diff(pg[c], pr[c])) <= 1e-12 * L and np.max(np.abs(vg[c] - vr[c])) <= 1e-12
    for a, r in zip(g.get_fields(), ref.get_fields()):
        assert np.linalg.norm(a - r) <= 1e-13 * max(np.linalg.norm(r), 1.0)


def test_tracers_are_refused_on_a_decomposed_context(MHD):
    """on a chunked context the push needs the slab stage (ooc_real_fields) to fill the tracers' copy of B, and
    that stage refuses a decomposed context.  Its return code is now propagated by mhd_tracers_push / mhd_step instead of
    being dropped; the one refusal reachable through the ABI is caught even earlier — mhd_tracers_bind rejects a
    decomposed context, so particles can never be pushed in a B array that was not written."""
    from paper_1810_12707_b200 import dist
    cfg = inputs.config1(32)
    grp = dist.Lockstep([dist.DistMHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt, rank=r, world=2) for r in range(2)])
    grp.set_fields(cfg.prim, "primitive")
    pos, vel = particles(64, 9)
    with pytest.raises(RuntimeError, match="decomposed"):
        grp.ranks[0].tracers_set(pos, vel)
    with pytest.raises(RuntimeError):
        grp.ranks[0].tracers_push(1)                     # nothing bound: refused, not MHD_OK


@pytest.mark.parametrize("every", [1, 3, 32])
def test_spatial_sort_does_not_change_results(MHD, every):
    """MHD_OPT_TRACER_SORT only reorders the particle storage: positions / velocities returned in id order are bitwise
    those of the unsorted run, for frozen pushes, stepping with the fields, and host or device output."""
    import torch
    cfg = inputs.config3(64, kmax=4)
    out = []
    for ev in (0, every):
        g = MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, 5e-3)
        g.set_option(11, ev)
        g.set_fields(cfg.prim, "primitive")
        pos, vel = particles(20011, 42, vscale=3.0)
        g.tracers_set(pos, vel)
        p0, v0 = g.tracers_get()
        for c in range(3):
            assert np.array_equal(p0[c], pos[c]) and np.array_equal(v0[c], vel[c])      # id order right after set
        g.tracers_push(7)
        g.step(5)
        g.tracers_push(2)
        ph, vh = g.tracers_get()
        pd, vd = g.tracers_get("device")
        for c in range(3):
            assert np.array_equal(pd[c].cpu().numpy(), ph[c]) and np.array_equal(vd[c].cpu().numpy(), vh[c])
        out.append((ph, vh))
    for c in range(3):
        assert np.array_equal(out[0][0][c], out[1][0][c]) and np.array_equal(out[0][1][c], out[1][1][c])


def test_bench_scale_256_both_B_sources_agree(MHD):
    """At the bench's 256^3 with 2 M tracers (the configuration `bench.py --tracers` times): B taken from the fused x
    sweep's by-product and B from the separate inverse transform move the particles identically to round-off, and the
    oracle's push on sampled particles reproduces one step."""
    import oracle
    cfg = inputs.config45(256)
    res = []
    for fused in (1, 2):
        g = MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt)
        g.set_option(1, fused)
        g.set_fields(cfg.prim, "primitive")
        pos, _ = particles(2_000_003, 77)
        g.tracers_set(pos)                       # v0 = CIC of u
        p0, v0 = g.tracers_get()
        if fused == 1:
            B = g.get_fields("conservative")[5:8]
            idx = np.arange(0, 2_000_003, 4001)
            ps, vs = oracle.tracers_push(B, [p[idx] for p in p0], [v[idx] for v in v0], cfg.dt, 1, L=cfg.L)
        g.step(4)
        res.append(g.tracers_get())
        if fused == 1:
            g2 = MHD(cfg.N, cfg.L, cfg.gamma, cfg.mu, cfg.eta, cfg.dt)
            g2.set_fields(cfg.prim, "primitive")
            g2.tracers_set(p0, v0)
            g2.step(1)
            p1, v1 = g2.tracers_get()
            for c in range(3):
                assert np.max(wrapped_diff(p1[c][idx], ps[c])) <= 1e-13 * L and np.max(np.abs(v1[c][idx] - vs[c])) <= 1e-13 * 10
            del g2
        del g
    for c in range(3):
        assert np.max(wrapped_diff(res[0][0][c], res[1][0][c])) <= 1e-12 * L
        assert np.max(np.abs(res[0][1][c] - res[1][1][c])) <= 1e-12 * 10
