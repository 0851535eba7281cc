"""GPU parity of the equation-set variants (include/mhd.h MHD_PARAM_CS2, MHD_PARAM_FORCE_AMP,
MHD_OPT_FORCE_K, MHD_OPT_EVOLVE) against the CPU oracle, through the C ABI.  Tolerances as in test_gpu_parity.py:
backward error beta_f <= 2e-15 per RHS field (plus the forcing scale f0 |rho| resp. f0 |m| in the denominator, which
is not under a derivative), state after n steps to 1e-12 of the largest field norm."""
import math

import numpy as np
import pytest

from paper_1810_12707_b200 import inputs

pytestmark = pytest.mark.gpu
NAMES = ["rho", "mx", "my", "mz", "E", "Bx", "By", "Bz"]


@pytest.fixture(scope="module")
def MHD():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1810_12707_b200 import build, binding
    build.build()
    return binding.MHD


def pair(orc, MHD, N, variant, mu=0.01, eta=0.02, dt=1e-3, flags=0, opts=None, seed=5):
    st = inputs.random_smooth_state(N, seed)
    o = orc.Oracle(N, 2 * math.pi, 5.0 / 3.0, mu, eta, dt)
    o.set_variant(**variant)
    o.set_fields(st, "primitive")
    g = MHD(N, 2 * math.pi, 5.0 / 3.0, mu, eta, dt, flags=flags)
    for k, v in (opts or {}).items():
        g.set_option(k, v)
    g.set_variant(**variant)
    g.set_fields(st, "primitive")
    return o, g


def check_rhs(o, g, N, f0=0.0):
    Ro, phi, dsc = o.rhs_scales()
    Rg = g.rhs()
    Uo = o.get_fields()
    kc = N // 3
    fscale = [0.0, f0 * np.linalg.norm(Uo[0]), f0 * np.linalg.norm(Uo[0]), f0 * np.linalg.norm(Uo[0]),
              f0 * max(np.linalg.norm(Uo[c]) for c in (1, 2, 3)), 0.0, 0.0, 0.0]
    for f in range(8):
        err = float(np.linalg.norm(Rg[f] - Ro[f]))
        scale = kc * phi[f] + kc * kc * dsc[f] + abs(fscale[f])
        if not np.any(Ro[f]):
            assert not np.any(Rg[f]), (NAMES[f], "switched-off equation must give exact zeros")
            continue
        assert err <= 2e-15 * scale, (NAMES[f], err / scale)


def check_state(o, g, tol=1e-12):
    Ug, Uo = g.get_fields(), o.get_fields()
    scale = max(np.linalg.norm(x) for x in Uo)
    for f in range(8):
        assert np.linalg.norm(Ug[f] - Uo[f]) <= tol * scale, NAMES[f]


@pytest.mark.parametrize("N,opts", [(32, None), (128, None), (128, {1: 2}), (32, {1: 0})])
def test_barotropic_closure(orc, MHD, N, opts):
    o, g = pair(orc, MHD, N, dict(cs2=1.3), opts=opts)
    check_rhs(o, g, N)
    n = 4 if N > 32 else 20
    o.step(n); g.step(n)
    check_state(o, g)
    # the energy field is carried, not evolved
    assert np.linalg.norm(g.get_fields()[4] - o.get_fields()[4]) <= 1e-12 * np.linalg.norm(o.get_fields()[4])


@pytest.mark.parametrize("N,kf,integ", [(32, 1, 0), (32, 3, 0), (128, 2, 0), (32, 2, 1), (32, 1, 2)])
def test_abc_forcing(orc, MHD, N, kf, integ):
    """mode-0 assembly (mhd_rhs, RK4 / PC stages) adds F^ after the assembly; the AB2 / Euler update reads it from a
    pre-pass: both against the oracle's real-space product rho f, m.f."""
    f0 = 0.7
    o, g = pair(orc, MHD, N, dict(f0=f0, kf=kf), opts={3: integ} if integ else None)
    check_rhs(o, g, N, f0)
    if integ == 0:
        n = 4 if N > 32 else 20
        o.step(n); g.step(n)
        check_state(o, g)
        check_rhs(o, g, N, f0)
    else:
        # RK4 / PC with forcing against AB2 with forcing over the same time with a much smaller step
        _, ga = pair(orc, MHD, N, dict(f0=f0, kf=kf), dt=1e-3 / 8)
        g.step(8); ga.step(64)
        Ua, Ug = ga.get_fields(), g.get_fields()
        scale = max(np.linalg.norm(x) for x in Ua)
        for f in range(8):
            assert np.linalg.norm(Ug[f] - Ua[f]) <= 2e-7 * scale, NAMES[f]


@pytest.mark.parametrize("evolve", [1, 2, 0])
def test_switched_off_equations(orc, MHD, evolve):
    N = 32
    o, g = pair(orc, MHD, N, dict(evolve=evolve))
    check_rhs(o, g, N)
    U0 = g.get_fields()
    o.step(10); g.step(10)
    check_state(o, g)
    U1 = g.get_fields()
    frozen = [c for c in range(8) if (c < 5 and not evolve & 1) or (c >= 5 and not evolve & 2)]
    for c in frozen:
        assert np.array_equal(U0[c], U1[c]), NAMES[c]


def test_kinematic_dynamo_with_forcing_and_barotropic_combined(orc, MHD):
    N = 32
    o, g = pair(orc, MHD, N, dict(cs2=0.9, f0=0.2, kf=1, evolve=3))
    check_rhs(o, g, N, 0.2)
    o.step(10); g.step(10)
    check_state(o, g)


def test_variants_on_the_chunked_pipeline(orc, MHD):
    from paper_1810_12707_b200 import binding as B
    N = 32
    for variant in (dict(cs2=1.1), dict(evolve=2)):
        o, g = pair(orc, MHD, N, variant, flags=B.MHD_FLAG_OUT_OF_CORE | B.MHD_FLAG_STATE_ON_HOST)
        check_rhs(o, g, N)
        o.step(5); g.step(5)
        check_state(o, g)
    g = MHD(N, flags=B.MHD_FLAG_OUT_OF_CORE)
    with pytest.raises(RuntimeError):
        g.set_param(2, 0.5)                       # forcing needs an in-core context
    g2 = MHD(N)
    with pytest.raises(RuntimeError):
        g2.set_param(1, -1.0)
    with pytest.raises(RuntimeError):
        g2.set_option(9, 0)
    with pytest.raises(RuntimeError):
        g2.set_option(8, 4)


def test_variant_change_resets_the_history(orc, MHD):
    """Like the oracle: changing a variant makes the next step a forward-Euler step."""
    N = 32
    o, g = pair(orc, MHD, N, dict())
    o.step(3); g.step(3)
    o.set_variant(f0=0.3, kf=2); g.set_variant(f0=0.3, kf=2)
    o.step(3); g.step(3)
    check_state(o, g)


# ---- MHD_OPT_STRESS: the viscous terms of Eq. 11-12 --------------------------------------------------------------------
def pair_stress(orc, MHD, N, mu=0.02, eta=0.01, dt=1e-3, opts=None, variant=None):
    st = inputs.random_smooth_state(N, 9)
    o = orc.Oracle(N, 2 * math.pi, 5.0 / 3.0, mu, eta, dt)
    o.set_stress(True)
    if variant:
        o.set_variant(**variant)
    o.set_fields(st, "primitive")
    g = MHD(N, 2 * math.pi, 5.0 / 3.0, mu, eta, dt)
    for k, v in (opts or {}).items():
        g.set_option(k, v)
    g.set_stress(True)
    if variant:
        g.set_variant(**variant)
    g.set_fields(st, "primitive")
    return o, g


@pytest.mark.parametrize("N,opts", [(32, None), (128, None), (64, {1: 0}), (128, {1: 2})])
def test_stress_tensor_variant(orc, MHD, N, opts):
    """Non-uniform density, compressive + solenoidal velocity: RHS (backward error; the viscous flux 2 nu rho S has one
    more derivative than the Laplacian form, covered by the k_c^2 d_f term) and the state after a few AB2 steps."""
    o, g = pair_stress(orc, MHD, N, opts=opts)
    check_rhs(o, g, N)
    n = 3 if N >= 128 else 10
    o.step(n); g.step(n)
    check_state(o, g)
    check_rhs(o, g, N)


def test_stress_tensor_with_forcing_and_tracers(orc, MHD):
    """The add-on pass shares the X / Y buffers with the forcing pre-pass and the tracers' real-space B: all three at once."""
    N = 32
    o, g = pair_stress(orc, MHD, N, variant=dict(f0=0.4, kf=2))
    rng = np.random.default_rng(1)
    pos = [rng.uniform(0, 2 * math.pi, 500) for _ in range(3)]
    vel = [rng.standard_normal(500) for _ in range(3)]
    o.tracers_set(pos, vel); g.tracers_set(pos, vel)
    check_rhs(o, g, N, 0.4)
    o.step(6); g.step(6)
    check_state(o, g)
    (po, vo), (pg, vg) = o.tracers_get(), g.tracers_get()
    for c in range(3):
        d = np.abs(pg[c] - po[c]); d = np.minimum(d, 2 * math.pi - d)
        assert np.max(d) <= 1e-12 and np.max(np.abs(vg[c] - vo[c])) <= 1e-12


def test_stress_tensor_restrictions(MHD):
    from paper_1810_12707_b200 import binding as B
    g = MHD(32)
    g.set_stress(True)
    g.set_option(3, 1)
    g.set_fields(inputs.random_smooth_state(32, 1), "primitive")
    with pytest.raises(RuntimeError):
        g.step(1)                                  # Adams-Bashforth only
    ooc = MHD(32, flags=B.MHD_FLAG_OUT_OF_CORE)
    with pytest.raises(RuntimeError):
        ooc.set_stress(True)
